"""sph_diagnostics_noalloc -- the one entry point for callers that cannot allocate device memory.

Some users of this library run inside a host program that owns the whole GPU (its particle pool took all the
memory at start-up, so a cudaMalloc for our workspace fails), or inside a loop where the device-wide stall of a
cudaMalloc is not acceptable.  For them the S8 conservation sums are available without context and workspace: the
partial sums sit in a static device array inside libsph.so.  The tests here check that this path gives what the
ordinary one (sph_get_diagnostics, partial sums in the caller's workspace) gives for the same particles, to the
1e-12 that test_diagnostics_match_fp64_sums_and_momentum_is_conserved uses, on two calls in a row that share the
static array, and that sizes beyond its capacity are refused.

The file name sorts last on purpose: pytest -x stops at the first failure, and a failure here should not hide the
parity tests.  It does not depend on them: it passes alone in a fresh process and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2603_19764_b200 import workloads as W

RTOL = 1e-12      # the tolerance of the existing diagnostics test (tests/test_gpu_parity.py)


def _moving(wl, salt):
    """Give the block seeded velocities and energies so that all eight sums are far from zero."""
    idx = np.arange(wl.n, dtype=np.uint64)
    for k, name in enumerate(("vx", "vy", "vz")):
        wl.arrays[name] = (100.0 * (W.uniform01(W.SEED_BASE + salt, idx, 40 + k) - 0.3)).astype(np.float32)
    wl.arrays["u"] = (1.0e4 * (1.0 + W.uniform01(W.SEED_BASE + salt, idx, 43))).astype(np.float32)
    return wl


def test_sizes_beyond_the_static_array_are_refused_and_bad_arguments_too():
    """No GPU needed: these are refused before any CUDA call."""
    from paper_2603_19764_b200 import binding as B
    lib = B.load()
    st = B.sph_state()
    dummy = (C.c_double * 8)()
    for k in ("x", "y", "z", "m", "vx", "vy", "vz", "u"):
        setattr(st, k, C.addressof(dummy))            # never dereferenced: the call returns before any launch
    err = C.c_int(-7)
    out = C.addressof(dummy)
    assert lib.sph_diagnostics_noalloc(C.byref(st), B.DIAG_NOALLOC_MAX_N + 1, out, None, C.byref(err)) == B.ECAPACITY
    assert err.value == 0
    assert lib.sph_diagnostics_noalloc(C.byref(st), -1, out, None, None) == B.EINVAL
    assert lib.sph_diagnostics_noalloc(None, 10, out, None, None) == B.EINVAL
    assert lib.sph_diagnostics_noalloc(C.byref(st), 10, None, None, None) == B.EINVAL
    st.vz = None
    assert lib.sph_diagnostics_noalloc(C.byref(st), 10, out, None, None) == B.EINVAL
    assert B.DIAG_NOALLOC_MAX_N == 1 << 25
    with pytest.raises(B.SphError, match="SPH_DIAG_NOALLOC_MAX_N"):
        class _T:                                     # stands in for a tensor: only data_ptr() / device are used
            device = None
            def data_ptr(self):
                return out
        class _S:
            cuda_stream = None
        B.diagnostics_noalloc({k: _T() for k in ("x", "y", "z", "m", "vx", "vy", "vz", "u")},
                              B.DIAG_NOALLOC_MAX_N + 1, _T(), stream=_S())


@pytest.mark.gpu
def test_no_alloc_sums_equal_the_workspace_path_on_two_calls_in_a_row():
    import torch
    from paper_2603_19764_b200 import binding as B
    # first a state that fills 16 rows of the static array (the last one ragged), then a smaller, different one that
    # fills 2: rows 2..15 of the first call are still in the array during the second and must not be read
    cases = [_moving(W.elastic_block(40), 1), _moving(W.elastic_block(17), 2)]
    assert cases[0].n == 64000 and cases[1].n == 4913
    expected, dev = [], []
    for wl in cases:                                   # the existing path: resident state, partials in the workspace
        s = B.Sph(wl.params, wl.n)
        t = s.upload(wl)
        s.build_neighbors(t, wl.n)
        expected.append(s.get_diagnostics().cpu().numpy())
        dev.append(t)
        s.close()
    outs = [torch.full((8,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    for wl, t, out in zip(cases, dev, outs):           # two calls back to back on one stream, no sync in between
        B.diagnostics_noalloc(t, wl.n, out)
    torch.cuda.synchronize()
    assert torch.cuda.memory_allocated() == before     # the wrapper allocated nothing either
    for wl, out, ref in zip(cases, outs, expected):
        got = out.cpu().numpy()
        assert np.all(np.isfinite(got)) and np.all(np.abs(ref) > 0)
        assert np.allclose(got, ref, rtol=RTOL, atol=RTOL * np.abs(ref).max()), (wl.n, got, ref)
    # and against plain fp64 sums of the same fp32 arrays
    A = {k: v.astype(np.float64) for k, v in cases[1].arrays.items()}
    m = A["m"]; x = np.stack([A["x"], A["y"], A["z"]]); v = np.stack([A["vx"], A["vy"], A["vz"]])
    ref = np.concatenate([[m.sum()], (m * v).sum(axis=1), (m * np.cross(x.T, v.T).T).sum(axis=1),
                          [(m * (0.5 * (v * v).sum(axis=0) + A["u"])).sum()]])
    assert np.allclose(outs[1].cpu().numpy(), ref, rtol=RTOL, atol=RTOL * np.abs(ref).max())
    # a fixed summation order: the same call again gives the same bits; n = 0 gives zeros
    again = torch.empty(8, dtype=torch.float64, device="cuda")
    B.diagnostics_noalloc(dev[0], cases[0].n, again)
    assert torch.equal(again, outs[0])
    B.diagnostics_noalloc(dev[0], 0, again)
    assert torch.equal(again, torch.zeros_like(again))
