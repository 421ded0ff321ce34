"""ck_source_terms_static: the source terms for callers that cannot allocate device memory.

Some users of this library run inside a solver whose own memory pool took the whole device at start-up,
or cannot afford the device-wide synchronisation that cudaMalloc and cudaFree bring into a time loop.
For them the library has one entry point whose scratch (the third-body concentrations M = C E of the
cells in flight) lives in a fixed 32 MiB array inside libck.so instead of in memory the handle
allocates.  That array is shared by every call and keeps the last call's contents, so the tests below
always make two calls in a row, of different sizes and on different states, and look at both results.
The reference is the library's existing path, ck_source_terms, on the same handle; the tolerance is the
north_star one every parity test here uses (helpers.parity_violations).

This file sorts last on purpose: pytest -x stops at the first failure, and a failure here must not hide
the parity tests.  It makes no assumption about what ran before it: it passes alone in a fresh process
(where its first call is the one that looks up the array's address) and after every other GPU test."""
import dataclasses

import numpy as np
import pytest

import ckgen
from helpers import parity_violations

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def ck():
    import paper_2008_08483_b200 as ck
    assert torch.cuda.is_available()
    return ck


def _device_state(cfg, N, seed_offset):
    dev = torch.device("cuda:0")
    T, P, Y = ckgen.states(cfg, N=N, seed_offset=seed_offset)
    put = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    return put(T), put(P), put(Y)


def _outputs(S, N):
    dev = torch.device("cuda:0")
    return (torch.full((S, N), float("nan"), dtype=torch.float64, device=dev),
            torch.full((N,), float("nan"), dtype=torch.float64, device=dev))


def _two_calls_in_a_row(gm, cfg, sizes, call):
    """Both calls are queued on one stream with no synchronisation in between (the second starts on
    the scratch the first one left); returns the results as numpy."""
    stream = torch.cuda.current_stream().cuda_stream
    runs = []
    for n, (N, so) in enumerate(zip(sizes, (11, 23))):
        T, P, Y = _device_state(cfg, N, so)
        w, d = _outputs(cfg.mech.S, N)
        runs.append((T, P, Y, w, d, N))
    for T, P, Y, w, d, N in runs:
        call(gm, T, P, Y, w, d, N, stream)
    torch.cuda.synchronize()
    return [(w.cpu().numpy(), d.cpu().numpy()) for _, _, _, w, d, _ in runs]


# the sizes span several tiles of 128 cells with a ragged tail; the first mid_1m size is larger than one
# wave of the kernel's grid, so a block's region of the array is reused from tile to tile within a call
CASES = [("tiny_1k", (70001, 1000)), ("mid_1m", (50001, 777)), ("large_256k", (3001, 20011))]


@pytest.mark.parametrize("cfg_name,sizes", CASES)
def test_static_scratch_matches_the_existing_path_on_two_calls_in_a_row(ck, cfg_name, sizes):
    cfg = ckgen.CONFIGS[cfg_name]
    with ck.Mechanism(ckgen.mechanism(cfg.mech)) as gm:
        new = _two_calls_in_a_row(gm, cfg, sizes, lambda g, T, P, Y, w, d, N, s: g.source_terms_static(T, P, Y, w, d, N=N, stream=s))
        old = _two_calls_in_a_row(gm, cfg, sizes, lambda g, T, P, Y, w, d, N, s: g.source_terms(T, P, Y, w, d, N=N, stream=s))
    for call, ((w, d), (wr, dr)) in enumerate(zip(new, old)):
        assert np.isfinite(wr).all() and np.isfinite(dr).all()
        rw, rt = parity_violations(w, d, wr, dr)
        assert rw <= 1.0, "%s call %d: wdot differs by %.3g x the tolerance" % (cfg_name, call, rw)
        assert rt <= 1.0, "%s call %d: dT/dt differs by %.3g x the tolerance" % (cfg_name, call, rt)


def test_handles_take_turns_on_the_one_array_and_nothing_is_allocated(ck):
    """Two mechanisms alternate on the shared array (each call finds the other's M values in it), and the
    device's free memory is the same after the calls as before them: the entry point allocated nothing.
    (Free memory is read after one warm-up call, which is where the CUDA runtime may load code.)"""
    stream = torch.cuda.current_stream().cuda_stream
    cfg_a, cfg_b = ckgen.CONFIGS["mid_1m"], ckgen.CONFIGS["tiny_1k"]
    with ck.Mechanism(ckgen.mechanism(cfg_a.mech)) as ga, ck.Mechanism(ckgen.mechanism(cfg_b.mech)) as gb:
        plan = [(ga, cfg_a, 4099, 1), (gb, cfg_b, 40000, 2), (ga, cfg_a, 300, 3), (gb, cfg_b, 129, 4)]
        bufs = []
        for gm, cfg, N, so in plan:
            T, P, Y = _device_state(cfg, N, so)
            bufs.append((gm, T, P, Y, N) + _outputs(cfg.mech.S, N) + _outputs(cfg.mech.S, N))
        gm, T, P, Y, N, w, d, _, _ = bufs[0]
        gm.source_terms_static(T, P, Y, w, d, N=N, stream=stream)
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        for gm, T, P, Y, N, w, d, _, _ in bufs:
            gm.source_terms_static(T, P, Y, w, d, N=N, stream=stream)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == free_before
        for gm, T, P, Y, N, _, _, wr, dr in bufs:
            gm.source_terms(T, P, Y, wr, dr, N=N, stream=stream)
        torch.cuda.synchronize()
    for i, (_, _, _, _, _, w, d, wr, dr) in enumerate(bufs):
        rw, rt = parity_violations(w.cpu().numpy(), d.cpu().numpy(), wr.cpu().numpy(), dr.cpu().numpy())
        assert rw <= 1.0 and rt <= 1.0, "call %d: %.3g / %.3g x the tolerance" % (i, rw, rt)


def test_same_bits_as_the_table_driven_kernel_it_is_a_variant_of(ck, monkeypatch):
    """The new kernel differs from the library's table-driven kernel (CK_KERNEL=generic) only in where
    M = C E is kept, so the two give the same bits."""
    monkeypatch.setenv("CK_KERNEL", "generic")
    cfg = ckgen.CONFIGS["mid_1m"]
    with ck.Mechanism(ckgen.mechanism(cfg.mech)) as gm:
        assert gm.info("jit") == 0
        new = _two_calls_in_a_row(gm, cfg, (40001, 515), lambda g, T, P, Y, w, d, N, s: g.source_terms_static(T, P, Y, w, d, N=N, stream=s))
        old = _two_calls_in_a_row(gm, cfg, (40001, 515), lambda g, T, P, Y, w, d, N, s: g.source_terms(T, P, Y, w, d, N=N, stream=s))
    for (w, d), (wr, dr) in zip(new, old):
        assert np.array_equal(w, wr) and np.array_equal(d, dr)


def test_sizes_beyond_the_static_array_and_unsupported_handles_are_refused(ck, monkeypatch):
    """More third-body reactions than the array has rows for (CK_STATIC_MAX_M_ROWS = 512): a clear error,
    nothing launched, outputs untouched.  The same for a handle whose rate layers exist only in the
    specialised kernel.  N = 0 stays a successful no-op."""
    stream = torch.cuda.current_stream().cuda_stream
    cfg = ckgen.CONFIGS["large_256k"]
    mech = ckgen.mechanism(cfg.mech)
    many = dataclasses.replace(mech, rxn_type=np.where(mech.rxn_type == 0, 1, mech.rxn_type).astype(np.uint8))
    assert int((many.rxn_type != 0).sum()) == 784 > 512
    T, P, Y = _device_state(cfg, 256, 5)
    w, d = _outputs(mech.n_species, 256)
    monkeypatch.setenv("CK_KERNEL", "generic")       # (no need to compile a specialised kernel for this)
    with ck.Mechanism(many) as gm:
        with pytest.raises(ck.CkError) as e:
            gm.source_terms_static(T, P, Y, w, d, N=256, stream=stream)
        assert e.value.status == 4 and "512" in str(e.value) and "784" in str(e.value)
        gm.source_terms_static(T, P, Y, w, d, N=0, stream=stream)
        gm.source_terms(T, P, Y, w, d, N=256, stream=stream)      # the allocating path still takes it
        torch.cuda.synchronize()
        assert torch.isfinite(w).all() and torch.isfinite(d).all()
    monkeypatch.delenv("CK_KERNEL")
    cfg = ckgen.CONFIGS["tiny_1k"]
    T, P, Y = _device_state(cfg, 256, 5)
    w, d = _outputs(cfg.mech.S, 256)
    with ck.Mechanism(ckgen.mechanism(cfg.mech), precision=ck.PREC_MIXED) as gm:
        with pytest.raises(ck.CkError) as e:
            gm.source_terms_static(T, P, Y, w, d, N=256, stream=stream)
        assert e.value.status == 4
    torch.cuda.synchronize()
    assert torch.isnan(w).all() and torch.isnan(d).all()
