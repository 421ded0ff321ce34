"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/ck.h
declares, and its argument validation (which runs before any CUDA call) returns the
documented status codes.  No compute calls here: those are the -m gpu tests."""
import ctypes
import dataclasses
import os
import re

import numpy as np
import pytest

import ckgen

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    return ck


def declared_functions():
    text = open(os.path.join(ROOT, "include", "ck.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(ck_[a-z0-9_]+)\s*\(", text)))


def test_header_declares_the_north_star_entry_points():
    names = declared_functions()
    for required in ("ck_mech_create", "ck_source_terms", "ck_mech_destroy"):
        assert required in names


def test_library_exports_every_declared_symbol(ck):
    lib = ctypes.CDLL(ck.library_path())
    for name in declared_functions():
        assert hasattr(lib, name), name


def test_binding_exposes_the_same_names(ck):
    for name in declared_functions():
        assert hasattr(ck, name), name


def test_product_does_not_import_the_oracle():
    """The product path never routes through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_2008_08483_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h", ".cuh", ".cpp")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src, f
                assert "ck_oracle" not in src, f


def test_create_rejects_invalid_mechanisms_before_touching_cuda(ck):
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    cases = [
        (dataclasses.replace(mech, mol_weight=-mech.mol_weight), 1),
        (dataclasses.replace(mech, T_mid=np.zeros(mech.n_species)), 1),
        (dataclasses.replace(mech, nu_reac=-mech.nu_reac), 1),
        (dataclasses.replace(mech, nu_prod=np.zeros_like(mech.nu_prod)), 1),
        (dataclasses.replace(mech, rxn_type=np.full(mech.n_reactions, 7, np.uint8)), 4),
        (dataclasses.replace(mech, p_ref=0.0), 1),
        (dataclasses.replace(mech, ln_A=np.full(mech.n_reactions, np.nan)), 1),
        (dataclasses.replace(mech, troe=-np.ones_like(mech.troe)), 1),
    ]
    for bad, status in cases:
        with pytest.raises(ck.CkError) as e:
            ck.Mechanism(bad)
        assert e.value.status == status, str(e.value)
        assert ck.ck_last_error() != ""


def test_source_terms_argument_checks_without_a_device(ck):
    with pytest.raises(ck.CkError) as e:
        ck.ck_source_terms(None, 8, 8, 8, 4, 8, 8)
    assert e.value.status == 1
    assert ck.ck_mech_info(None, 0) == -1
    ck.ck_mech_destroy(None)      # NULL is a no-op


def test_binding_checks_shapes(ck):
    mech = ckgen.mechanism(ckgen.MECH_TINY)
    with pytest.raises(ValueError):
        ck.Mechanism(dataclasses.replace(mech, troe=mech.troe[:, :3]))
