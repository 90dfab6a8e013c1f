"""GPU test of tm_field_redot_noalloc (include/tm.h): Re <x, y> with its scratch in a fixed __device__ array, for callers that may
not call cudaMalloc (graph capture, serving loops).  Checked against the existing path, tm_field_redot, on two calls in a row.

Collected last on purpose (the suite runs with pytest -x: a failure here must not hide the other tests); passes alone in a
fresh process and after the rest of the suite (the first call on a device looks up the array's address, later calls reuse it).
"""
import numpy as np
import pytest

import paper_1311_4462_b200 as tm
import synth_inputs as si

pytestmark = pytest.mark.gpu

# the two paths add the same double-precision products in the same order (csrc/tm_noalloc.cu): they agree bit for bit; the bound
# used is the double-precision one of test_s1 in test_gpu_solver.py (1e-13 x 10 x |x| |y|), far below any precision's storage error
RTOL = 1e-12


def both(lat, fx, fy, out):
    """(existing path, new entry point) for one pair of fields; `out` is the caller's device double"""
    want = tm.field_redot(fx, fy)
    out.fill_(float("nan"))
    tm.tm_field_redot_noalloc(fx.h, fy.h, out.data_ptr())
    lat.sync()
    return want, float(out.item())


@pytest.mark.parametrize("nf", [1, 2])
def test_z1_redot_noalloc_matches_redot_on_two_calls_in_a_row(nf):
    import torch
    # first call: 16^3 x 32 (512 partial sums); second call: 6^4 (6 partial sums, ragged last tile) on a context of its own -- the
    # scratch array still holds the first call's 512 sums and none of them may leak into the second result
    big, small = (16, 16, 16, 32), (6, 6, 6, 6)
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    lat_b, lat_s = tm.Lattice(big), tm.Lattice(small)
    xb = si.mask_parity(si.spinor_field(big, nf, 41), big, 0)
    yb = si.mask_parity(si.spinor_field(big, nf, 42), big, 0)
    xs = si.mask_parity(si.spinor_field(small, nf, 43), small, 0)
    ys = si.mask_parity(si.spinor_field(small, nf, 44), small, 0)
    for prec, tol in ((tm.TM_DOUBLE, 1e-13), (tm.TM_SINGLE, 1e-6), (tm.TM_HALF, 2e-4)):
        fxb, fyb = lat_b.field(prec, nf).upload(0, xb), lat_b.field(prec, nf).upload(0, yb)
        fxs, fys = lat_s.field(prec, nf).upload(0, xs), lat_s.field(prec, nf).upload(0, ys)
        n0 = lat_b.launches()
        w1, g1 = both(lat_b, fxb, fyb, out)                 # call 1
        w2, g2 = both(lat_s, fxs, fys, out)                 # call 2, right after it, smaller
        w3, g3 = both(lat_b, fxb, fxb, out)                 # and back: |x|^2 on the large lattice
        scale_b = np.linalg.norm(xb) * np.linalg.norm(yb)
        assert abs(g1 - w1) <= RTOL * scale_b, (prec, g1, w1)
        assert abs(g2 - w2) <= RTOL * np.linalg.norm(xs) * np.linalg.norm(ys), (prec, g2, w2)
        assert abs(g3 - w3) <= RTOL * np.linalg.norm(xb) ** 2, (prec, g3, w3)
        # and the existing path itself against numpy, at the storage precision's tolerance (as test_s1): the comparison above is not
        # between two wrong numbers
        assert abs(w1 - np.vdot(xb, yb).real) <= tol * 10 * scale_b
        assert abs(g3 - np.vdot(xb, xb).real) <= tol * 10 * np.vdot(xb, xb).real
        assert lat_b.launches() - n0 == 4                   # 2 calls of each path on this context, one counted launch each


def test_z2_redot_noalloc_rejects_what_its_scratch_cannot_hold_and_bad_arguments():
    import torch
    out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    dims = (64, 64, 64, 66)                                 # 8 650 752 sites per parity > TM_NOALLOC_MAX_SITES = 8 388 608
    lat = tm.Lattice(dims)
    assert lat.Vh > tm.TM_NOALLOC_MAX_SITES
    f = lat.field(tm.TM_HALF, 1)                            # 450 MB; never read: the call is refused before any launch
    n0 = lat.launches()
    with pytest.raises(tm.TmError) as e:
        tm.tm_field_redot_noalloc(f.h, f.h, out.data_ptr())
    assert "TM_NOALLOC_MAX_SITES" in str(e.value) and str(lat.Vh) in str(e.value)
    assert lat.launches() == n0
    del f
    lat = tm.Lattice((8, 8, 8, 8))
    fd, fs, f2 = lat.field(tm.TM_DOUBLE, 1), lat.field(tm.TM_SINGLE, 1), lat.field(tm.TM_DOUBLE, 2)
    with pytest.raises(tm.TmError):
        tm.tm_field_redot_noalloc(fd.h, fs.h, out.data_ptr())          # precision mismatch
    with pytest.raises(tm.TmError):
        tm.tm_field_redot_noalloc(fd.h, f2.h, out.data_ptr())          # flavor mismatch
    with pytest.raises(tm.TmError):
        tm.tm_field_redot_noalloc(fd.h, fd.h, 0)                       # NULL result pointer
