"""aton_field_sums_noalloc (include/aton.h): the two-pass diagnostic reduction with its scratch in a static __device__
array -- no cudaMalloc, no context, no synchronisation -- against the existing path (aton_reduce_sums of a context that
holds the same fields), on two calls in a row that share the static array.  The file sorts last on purpose: the suite
runs with pytest -x, and a failure here must not hide the tests before it."""
import numpy as np
import pytest
import torch

from paper_1004_2503_b200 import workloads as wl

pytestmark = pytest.mark.gpu

# (index in aton_field_sums_noalloc's sums, index in aton_reduce_sums' sums, relative tolerance).  The sums are fp64
# accumulations of the same fp32 values in the same order (same block count, same row order): 1e-12; max f is formed from F
# here and from G = F/c rounded to fp32 in the context: the 1e-6 of test_reduce_matches_oracle.
PAIRS = [(0, 0, 0.0), (1, 1, 1e-12), (2, 2, 1e-12), (3, 3, 1e-12), (4, 4, 1e-12), (5, 5, 1e-12), (6, 6, 1e-12),
         (7, 7, 0.0), (8, 8, 0.0), (9, 11, 1e-6), (10, 13, 0.0)]


def _state(n, seed):
    """A seeded mid-reionisation state on an n^3 twin of config 4 (bubbles, photons, |F| <= 0.9 cN)."""
    w = wl.synthetic_warm_state(wl.make_config(4, n=n, device="cuda"), seed=seed)
    return w, [t.contiguous() for t in w.fields()]          # nH, x, T, N, Fx, Fy, Fz


def _existing_path(w, f):
    from paper_1004_2503_b200 import aton
    a = aton.Aton(w.n, w.n, w.n, w.box_cm, w.params)
    a.set_fields(*f)
    sums = a.reduce_sums()
    a.close()
    return sums


def test_noalloc_sums_equal_the_context_path_on_two_calls_in_a_row():
    from paper_1004_2503_b200 import aton
    # the second call is SMALLER than the first: the static array still holds rows of the first call beyond the ones the
    # second one writes -- they must not be read
    cases = [_state(96, 11), _state(32, 12)]
    outs = [torch.full((aton.NOALLOC_NSUMS,), float("nan"), dtype=torch.float64, device="cuda") for _ in cases]
    before = torch.cuda.memory_allocated()
    for (w, f), out in zip(cases, outs):                    # back to back on one stream, no synchronisation in between
        aton.field_sums_noalloc(*f, out=out, c_cm_s=w.params["c_cm_s"])
    assert torch.cuda.memory_allocated() == before          # (torch's view: the binding made no tensor either)
    torch.cuda.synchronize()
    for (w, f), out in zip(cases, outs):
        got = out.cpu().numpy()
        ref = _existing_path(w, f)
        assert np.all(np.isfinite(got)) and got[0] == w.n ** 3 and got[4] > 0 and got[8] == 0
        for i, j, rel in PAIRS:
            assert got[i] == pytest.approx(ref[j], rel=rel, abs=0.0), (w.n, i, j, got[i], ref[j])
        assert got[11] == pytest.approx(float(f[0].min()), rel=0, abs=0)         # min n_H: exact
    # and once more on the first case: the same numbers, bit for bit (deterministic, nothing left over from call two)
    again = torch.empty_like(outs[0])
    aton.field_sums_noalloc(*cases[0][1], out=again, c_cm_s=cases[0][0].params["c_cm_s"])
    torch.cuda.synchronize()
    assert torch.equal(again, outs[0])


def test_noalloc_rejects_what_it_cannot_take():
    from paper_1004_2503_b200 import aton
    L = aton.load_library()
    import ctypes as C
    f = [torch.ones(64, device="cuda") for _ in range(7)]
    out = torch.zeros(aton.NOALLOC_NSUMS, dtype=torch.float64, device="cuda")
    p = [C.c_void_p(t.data_ptr()) for t in f]
    o = C.c_void_p(out.data_ptr())
    assert L.aton_field_sums_noalloc(*p, 64, 0.0, None, o) == aton.OK
    assert L.aton_field_sums_noalloc(*p, 1 << 31, 0.0, None, o) == aton.EINVAL               # beyond the stated maximum
    assert "maximum" in L.aton_last_error(None).decode()
    assert L.aton_field_sums_noalloc(*p, 62, 0.0, None, o) == aton.EINVAL                    # not a multiple of 4
    assert L.aton_field_sums_noalloc(*p, 0, 0.0, None, o) == aton.EINVAL
    assert L.aton_field_sums_noalloc(None, *p[1:], 64, 0.0, None, o) == aton.EINVAL
    assert L.aton_field_sums_noalloc(*p, 64, 0.0, None, None) == aton.EINVAL
    q = list(p); q[2] = C.c_void_p(f[2].data_ptr() + 4)                                       # misaligned
    assert L.aton_field_sums_noalloc(*q, 60, 0.0, None, o) == aton.EINVAL
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert got[0] == 64 and got[1] == 64 and got[3] == 64 and got[7] == 64 and got[11] == 1.0
