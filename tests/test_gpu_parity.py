"""GPU parity tests: every C-ABI entry point against the CPU oracle, element by element, on seeded inputs.

Tolerances are BASELINE.json's: relative L2 over the whole output parity field (both flavors together)
<= 1e-12 (double), 1e-5 (single), 5e-3 (half).  Half inputs are quantised by the library on upload; the oracle
always sees the unquantised double inputs (reading C9, primary comparison).
"""
import itertools

import numpy as np
import pytest

import oracle
import paper_1311_4462_b200 as tm
import synth_inputs as si
from gpu_util import TOL, PREC_NAME, Bench, rel_l2

pytestmark = pytest.mark.gpu

KAPPA = 0.1632
PRECS = [tm.TM_DOUBLE, tm.TM_SINGLE, tm.TM_HALF]
RECONS = [tm.TM_RECON_18, tm.TM_RECON_12]
FLAVORS = [
    dict(mu=0.004, epsilon=0.0, twist_flavor=1),
    dict(mu=0.3, epsilon=0.0, twist_flavor=-1),
    dict(mu=0.15, epsilon=0.19, twist_flavor=0),
]


# code paths of the library: (id, tm_set_path, tm_set_tuning overrides); results must not depend on them
VARIANTS = [
    ("default", 0, {}),
    ("scalar", 1, {}),
    ("packed-direct", 0, {"stage_links": 0, "block_threads": 128}),
    ("packed-staged", 0, {"stage_links": 1, "block_threads": 64, "prefetch_blocks": 3}),
    ("scalar-staged", 1, {"stage_links": 1, "block_threads": 32}),
]


def nf_of(kw):
    return 2 if kw["twist_flavor"] == 0 else 1


_cache = {}


def bench_for(dims, kind, seed):
    key = (tuple(dims), kind, seed)
    if key not in _cache:
        _cache[key] = Bench(dims, si.gauge_field(dims, seed, kind))
    ctx = _cache[key].lat.ctx                       # default kernel selection unless a test asks otherwise
    tm.tm_set_path(ctx, 0)
    tm.tm_set_tuning(ctx, "stage_links", -1)
    tm.tm_set_tuning(ctx, "block_threads", 0)
    tm.tm_set_tuning(ctx, "prefetch_blocks", -1)
    tm.tm_set_tuning(ctx, "z_chunks", -1)
    tm.tm_set_tuning(ctx, "tile_kernel", -1)
    tm.tm_set_tuning(ctx, "pdl", 1)
    return _cache[key]


# ---- T1: layouts round trip -----------------------------------------------------------------------

# (6, 6, 6, 6): V/2 = 648 sites = 20.25 tiles of 32 (ragged last tile), X/2 = 3 (no power-of-two extents)
@pytest.mark.parametrize("dims", [(4, 4, 4, 8), (4, 6, 8, 10), (6, 6, 6, 6)])
@pytest.mark.parametrize("nf", [1, 2])
def test_t1_spinor_pack_unpack_round_trip(dims, nf):
    lat = tm.Lattice(dims)
    psi = si.spinor_field(dims, nf, 5)
    for prec in PRECS:
        for parity in (0, 1):
            f = lat.field(prec, nf).upload(parity, psi)
            back = f.download(parity)
            want = si.mask_parity(psi, dims, parity)
            assert np.abs(si.mask_parity(back, dims, 1 - parity)).max() == 0
            if prec == tm.TM_DOUBLE:
                assert np.array_equal(back, want)
            elif prec == tm.TM_SINGLE:
                assert np.array_equal(back, want.astype(np.complex64).astype(np.complex128))
            else:
                # <= 1/2 LSB of the site's scale: |v - deq| <= 0.5 * norm / 32767 (+ fp32 rounding)
                idx = si.parity_sites(dims, parity)
                w = want[:, idx].reshape(nf, len(idx), 24 // 2)
                b = back[:, idx].reshape(nf, len(idx), 24 // 2)
                norm = np.maximum(np.abs(w.real).max(axis=2), np.abs(w.imag).max(axis=2))[..., None]
                err = np.maximum(np.abs((w - b).real), np.abs((w - b).imag))
                assert (err <= (0.5 / 32767 + 1e-6) * norm).all()     # 1e-6: fp32 rounding of the scale
            # the cb entry points see the same field
            cb = f.download_cb(parity)
            assert np.array_equal(cb, back[:, si.parity_sites(dims, parity)])
            g = lat.field(prec, nf).upload_cb(parity, si.to_parity(psi, dims, parity))
            assert np.array_equal(g.download(parity), back)


def test_t1b_async_transfers_overlap_safely():
    """tm_field_upload_cb_async / tm_field_download_cb_async: a chain of composites that reuses the same device fields
    (upload k+1 overwrites the input of composite k, composite k+1 overwrites the output being downloaded) gives
    bit-identical results to the synchronous entry points."""
    import torch
    dims = (8, 8, 8, 16)
    bench = bench_for(dims, "haar", 9)
    lat = bench.lat
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    pg = tm.params(KAPPA, **kw)
    n = 2 * lat.Vh * 24
    ins = [si.to_parity(si.spinor_field(dims, 2, 70 + k), dims, 0) for k in range(4)]
    for prec in PRECS:
        g = bench.gauge(prec, tm.TM_RECON_12)
        fin, ftmp, fout = lat.field(prec, 2), lat.field(prec, 2), lat.field(prec, 2)
        want = []
        for a in ins:                                              # synchronous reference
            fin.upload_cb(0, a)
            tm.mat_pc(fout, fin, ftmp, g, pg, tm.TM_MATPC_SYM, 0)
            want.append(fout.download_cb(0).copy())
        pin_in = [torch.empty(n, dtype=torch.float64, pin_memory=True) for _ in ins]
        pin_out = [torch.zeros(n, dtype=torch.float64, pin_memory=True) for _ in ins]
        for t, a in zip(pin_in, ins):
            t.numpy()[:] = a.view(np.float64).reshape(-1)
        for k in range(len(ins)):
            tm.tm_field_upload_cb_async(fin.h, 0, pin_in[k].data_ptr())
            tm.mat_pc(fout, fin, ftmp, g, pg, tm.TM_MATPC_SYM, 0)
            tm.tm_field_download_cb_async(fout.h, 0, pin_out[k].data_ptr())
        lat.sync()
        for k in range(len(ins)):
            got = pin_out[k].numpy().view(np.complex128).reshape(want[k].shape)
            assert np.array_equal(got, want[k]), (PREC_NAME[prec], k)


def test_t1c_float_host_arrays_round_trip():
    """tm_field_upload_cb_async_f32 / tm_field_download_cb_async_f32: float host arrays (half the PCIe bytes for single and half
    fields).  Round trip: exact for a single field, float rounding for a double field, 1/2 LSB of the site norm for a half field;
    and the uploaded field equals the one uploaded from the double array (single, half: bit for bit)."""
    import torch
    dims, nf = (6, 6, 6, 6), 2
    lat = tm.Lattice(dims)
    vh = lat.Vh
    x = si.to_parity(si.spinor_field(dims, nf, 9), dims, 0)
    x32 = x.view(np.float64).astype(np.float32)
    pin = torch.empty(x32.size, dtype=torch.float32, pin_memory=True)
    pin.numpy()[:] = x32.reshape(-1)
    back = torch.zeros(x32.size, dtype=torch.float32, pin_memory=True)
    for prec in PRECS:
        f, fd = lat.field(prec, nf), lat.field(prec, nf)
        tm.tm_field_upload_cb_async_f32(f.h, 0, pin.data_ptr())
        tm.tm_field_download_cb_async_f32(f.h, 0, back.data_ptr())
        lat.sync()
        got = back.numpy().reshape(nf, vh, 24)
        want = x32.reshape(nf, vh, 24)
        if prec == tm.TM_HALF:
            lsb = np.abs(got - want) / (np.abs(want).max(axis=2, keepdims=True) / 32767.0)
            assert lsb.max() <= 0.51, lsb.max()
        else:
            assert np.array_equal(got, want)
        fd.upload_cb(0, x32.astype(np.float64).view(np.complex128).reshape(nf, vh, 4, 3))      # the same values through the double entry point
        lat.sync()
        assert bool((f.storage == fd.storage).all()), prec


# ---- T2: every kernel variant vs the oracle -------------------------------------------------------

@pytest.mark.parametrize("dims,kind", [((4, 4, 4, 8), "haar"), ((4, 6, 8, 10), "near_identity"), ((8, 4, 6, 4), "haar"),
                                       ((6, 6, 6, 6), "haar")])
@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
@pytest.mark.parametrize("variant", VARIANTS, ids=[v[0] for v in VARIANTS])
def test_t2_every_kernel_variant_matches_oracle(dims, kind, kw, variant):
    nf = nf_of(kw)
    bench = bench_for(dims, kind, 1)
    tm.tm_set_path(bench.lat.ctx, variant[1])
    for key, val in variant[2].items():
        tm.tm_set_tuning(bench.lat.ctx, key, val)
    po = oracle.params(dims, KAPPA, **kw)
    pg = tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 2), si.spinor_field(dims, nf, 3)
    worst = {}
    for parity, dagger, kt in itertools.product((0, 1), (0, 1), (0, 1, 2, 3)):
        inp = si.mask_parity(full_in, dims, 1 - parity)
        x = si.mask_parity(full_x, dims, parity)
        want = oracle.kernel(inp, x, bench.U, po, parity, dagger, kt)
        for prec, recon in itertools.product(PRECS, RECONS):
            got = bench.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, prec, recon, nf)
            err = rel_l2(got, want)
            worst[prec] = max(worst.get(prec, 0.0), err)
            assert err <= TOL[prec], (PREC_NAME[prec], recon, parity, dagger, kt, err)
            assert np.abs(si.mask_parity(got, dims, 1 - parity)).max() == 0
    print("worst rel L2:", {PREC_NAME[k]: v for k, v in worst.items()})


@pytest.mark.parametrize("kw", [FLAVORS[0], FLAVORS[2]], ids=["deg", "ndeg"])
@pytest.mark.parametrize("chunks,threads", [(2, 128), (4, 64), (8, 32)])
def test_t2e_z_chunked_traversal_matches_oracle(kw, chunks, threads):
    """tm_set_tuning("z_chunks"): the thread blocks walk the lattice chunk by chunk of Z / n z-planes (the library turns this on
    by itself when three time slices of the input do not fit the L2, e.g. 48^3 x 96 fp64 doublet).  A permutation of the block
    order only: every kernel type must still match the oracle.  16 x 8 x 16 x 6: 1024 sites per slice and parity."""
    dims, nf = (16, 8, 16, 6), nf_of(kw)
    bench = bench_for(dims, "haar", 6)
    tm.tm_set_tuning(bench.lat.ctx, "z_chunks", chunks)
    tm.tm_set_tuning(bench.lat.ctx, "block_threads", threads)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 2), si.spinor_field(dims, nf, 3)
    for parity, dagger, kt in ((0, 0, 0), (1, 1, 1), (0, 1, 2), (1, 0, 3)):
        inp, x = si.mask_parity(full_in, dims, 1 - parity), si.mask_parity(full_x, dims, parity)
        want = oracle.kernel(inp, x, bench.U, po, parity, dagger, kt)
        for prec in PRECS:
            got = bench.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, prec, tm.TM_RECON_12, nf)
            assert rel_l2(got, want) <= TOL[prec], (PREC_NAME[prec], parity, dagger, kt, rel_l2(got, want))
    for path in (0, 1):                      # packed and scalar kernels
        tm.tm_set_path(bench.lat.ctx, path)
        inp = si.mask_parity(full_in, dims, 0)
        want = oracle.matpc(inp, bench.U, po, oracle.SYM, 0)
        got = bench.matpc(inp, pg, tm.TM_MATPC_SYM, 0, tm.TM_SINGLE, tm.TM_RECON_18, nf)
        assert rel_l2(got, want) <= TOL[tm.TM_SINGLE]


@pytest.mark.parametrize("dims", [(8, 8, 4, 4), (16, 4, 4, 4), (16, 8, 4, 6), (32, 4, 4, 4), (32, 6, 4, 4)],
                         ids=["Xh4-1tile-per-slab", "Xh8-1", "Xh8-2", "Xh16-2", "Xh16-3"])
@pytest.mark.parametrize("kw", [FLAVORS[1], FLAVORS[2]], ids=["deg-", "ndeg"])
def test_t2f_warp_per_tile_half_kernel_matches_oracle(dims, kw):
    """The warp-per-tile half-precision kernel (tm_dslash_tile.cuh: every operand staged through shared memory, neighbours addressed
    by slot) on the lattices it covers -- X/2 in {4, 8, 16}, one, two and three tiles per (z, t) slab, so that the y-wrap inside one
    tile, between two tiles and across the slab are all exercised -- against the oracle: every kernel type, parity, dagger, link
    compression; and bit-identical to the thread-per-site packed kernel (same arithmetic, different data path)."""
    nf = nf_of(kw)
    bench = bench_for(dims, "haar", 5)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 2), si.spinor_field(dims, nf, 3)
    for parity, dagger, kt in itertools.product((0, 1), (0, 1), (0, 1, 2, 3, 4, 5)):
        inp, x = si.mask_parity(full_in, dims, 1 - parity), si.mask_parity(full_x, dims, parity)
        want = oracle.kernel(inp, x, bench.U, po, parity, dagger, kt) if kt < 4 else \
            oracle.hop_xpay(inp, x, bench.U, po, parity, dagger, -KAPPA ** 2 if kt == 4 else KAPPA)
        for recon in RECONS:
            tm.tm_set_tuning(bench.lat.ctx, "tile_kernel", 1)          # (the default where the geometry fits)
            got = bench.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, tm.TM_HALF, recon, nf)
            assert tm.tm_last_kernel_name(bench.lat.ctx).startswith("tile<"), tm.tm_last_kernel_name(bench.lat.ctx)
            assert rel_l2(got, want) <= TOL[tm.TM_HALF], (recon, parity, dagger, kt, rel_l2(got, want))
            tm.tm_set_tuning(bench.lat.ctx, "tile_kernel", 0)
            ref = bench.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, tm.TM_HALF, recon, nf)
            assert tm.tm_last_kernel_name(bench.lat.ctx).startswith("f2")
            assert np.array_equal(got, ref), (recon, parity, dagger, kt, np.abs(got - ref).max())
    tm.tm_set_tuning(bench.lat.ctx, "tile_kernel", -1)


def test_t2b_periodic_time_and_wilson_limit():
    dims = (4, 4, 6, 8)
    bench = bench_for(dims, "haar", 7)
    for kw in (dict(mu=0.0, epsilon=0.0, twist_flavor=1, t_boundary=+1), dict(mu=0.0, epsilon=0.0, twist_flavor=0, t_boundary=-1),
               dict(mu=0.15, epsilon=0.19, twist_flavor=0, t_boundary=+1)):
        nf = nf_of(kw)
        po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
        inp = si.mask_parity(si.spinor_field(dims, nf, 8), dims, 0)
        x = si.mask_parity(si.spinor_field(dims, nf, 9), dims, 1)
        for kt in (0, 1, 2, 3):
            want = oracle.kernel(inp, x, bench.U, po, 1, 0, kt)
            for prec in PRECS:
                got = bench.kernel(inp, x, pg, 1, 0, kt, prec, tm.TM_RECON_12, nf)
                assert rel_l2(got, want) <= TOL[prec]


# ---- T2d: half precision, tight comparison (reading C9, secondary comparison) ---------------------------------

def _quantise_spinor(a):
    """The half format of reading C9 written out in numpy (fp32, as the library stores it): per (flavor, site) norm = max |v_i|
    over the 24 reals, q = rint(v * 32767 / norm), value = q * norm / 32767.  Nothing here comes from the CUDA path."""
    v = a.view(np.float64).reshape(a.shape[0], a.shape[1], 24).astype(np.float32)
    m = np.abs(v).max(axis=2, keepdims=True)
    s = np.where(m > 0, np.float32(32767.0) / np.where(m > 0, m, np.float32(1)), np.float32(0)).astype(np.float32)
    q = np.rint(v * s).astype(np.float32)
    deq = (q * (m * np.float32(1.0 / 32767.0))).astype(np.float64)
    return deq.reshape(a.shape[0], a.shape[1], 4, 3, 2).view(np.complex128).reshape(a.shape)


def _quantise_links(U):
    """Half gauge field, 18-real: q = rint(u * 32767) at fixed scale, no norms."""
    r = U.view(np.float64).astype(np.float32)
    q = np.rint(r * np.float32(32767.0)).astype(np.float32)
    return (q.astype(np.float64) / 32767.0).view(np.complex128).reshape(U.shape)


@pytest.mark.parametrize("dims,kind", [((4, 6, 8, 10), "near_identity"), ((6, 6, 6, 6), "haar")])
@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
def test_t2d_half_against_the_oracle_on_the_quantised_inputs(dims, kind, kw):
    """The primary half comparison (T2) allows 5e-3 because the oracle sees the unquantised inputs.  Here the oracle is fed
    the inputs AS STORED (quantised in numpy by the definition of the format), so what is left is the fp32 arithmetic and the
    quantisation of the output, <= 1/2 LSB of the site norm: two orders tighter, enough to see a scale of 32768 for 32767."""
    nf = nf_of(kw)
    bench = bench_for(dims, kind, 1)
    Uq = _quantise_links(bench.U)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 16), si.spinor_field(dims, nf, 17)
    worst = 0.0
    for parity, dagger, kt in itertools.product((0, 1), (0, 1), (0, 1, 2, 3)):
        inp = si.mask_parity(full_in, dims, 1 - parity)
        x = si.mask_parity(full_x, dims, parity)
        want = oracle.kernel(_quantise_spinor(inp), _quantise_spinor(x), Uq, po, parity, dagger, kt)
        got = bench.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, tm.TM_HALF, tm.TM_RECON_18, nf)
        err = rel_l2(got, want)
        worst = max(worst, err)
        assert err <= 5e-5, (parity, dagger, kt, err)
        # component-wise, in LSB of the site norm (from the oracle): the output quantisation is 1/2 LSB; an input value that sits
        # on a rounding tie may be stored one LSB away from the numpy model (the library rounds v * s in one FMA), which the
        # xpay forms pass straight to the output -- so: almost all components within 0.7 LSB, none beyond 1.75
        idx = si.parity_sites(dims, parity)
        w = want[:, idx].view(np.float64).reshape(nf, len(idx), 24)
        g = got[:, idx].view(np.float64).reshape(nf, len(idx), 24)
        lsb = np.abs(g - w) / (np.abs(w).max(axis=2, keepdims=True) / 32767.0 + 1e-300)
        assert lsb.max() <= 1.75, (parity, dagger, kt, lsb.max())
        assert (lsb > 0.7).mean() <= 0.02, (parity, dagger, kt, (lsb > 0.7).mean())
    print("worst rel L2 (half, quantised inputs):", worst)


# ---- T2c: 8-real links ------------------------------------

@pytest.mark.parametrize("dims,kind", [((4, 4, 4, 8), "haar"), ((4, 6, 8, 10), "near_identity"), ((6, 6, 6, 6), "haar")])
@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
def test_t2c_recon8_every_kernel_matches_oracle(dims, kind, kw):
    """The oracle multiplies the full 18-real double links; the library stores 8 reals per link and rebuilds the
    matrix in the kernel, so this checks the chart, its packing and the rebuild in all three precisions."""
    nf = nf_of(kw)
    bench = bench_for(dims, kind, 1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 12), si.spinor_field(dims, nf, 13)
    worst = {}
    for parity, dagger, kt in itertools.product((0, 1), (0, 1), (0, 1, 2, 3)):
        inp = si.mask_parity(full_in, dims, 1 - parity)
        x = si.mask_parity(full_x, dims, parity)
        want = oracle.kernel(inp, x, bench.U, po, parity, dagger, kt)
        for prec in PRECS:
            got = bench.kernel(inp, None if kt == 0 else x, pg, parity, dagger, kt, prec, tm.TM_RECON_8, nf)
            assert ",8," in tm.tm_last_kernel_name(bench.lat.ctx)
            err = rel_l2(got, want)
            worst[prec] = max(worst.get(prec, 0.0), err)
            assert err <= TOL[prec], (PREC_NAME[prec], parity, dagger, kt, err)
    print("worst rel L2 (8-real):", {PREC_NAME[k]: v for k, v in worst.items()})


def test_t2c_recon8_composites_and_singular_chart():
    dims = (4, 4, 6, 8)
    bench = bench_for(dims, "haar", 7)
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi_e = si.mask_parity(si.spinor_field(dims, 2, 14), dims, 0)
    b_o = si.mask_parity(si.spinor_field(dims, 2, 15), dims, 1)
    for prec in PRECS:
        for typ, dagger in ((tm.TM_MATPC_ASYM, 0), (tm.TM_MATPC_ASYM, 1), (tm.TM_MATPC_SYM, 0), (tm.TM_MATPC_SYM, 1)):
            want = oracle.matpc_adjoint(psi_e, bench.U, po, typ) if dagger else oracle.matpc(psi_e, bench.U, po, typ, 0)
            assert rel_l2(bench.matpc(psi_e, pg, typ, dagger, prec, tm.TM_RECON_8, 2), want) <= TOL[prec], (PREC_NAME[prec], typ, dagger)
        want = oracle.reconstruct_odd(psi_e, b_o, bench.U, po)
        assert rel_l2(bench.reconstruct_odd(psi_e, b_o, pg, prec, tm.TM_RECON_8, 2), want) <= TOL[prec]
    # the unit matrix sits on the chart's singular point: refused at load time, not NaN at run time
    unit = np.zeros((4, bench.lat.V, 3, 3), dtype=np.complex128)
    unit[:, :, [0, 1, 2], [0, 1, 2]] = 1.0
    with pytest.raises(tm.TmError) as ei:
        bench.lat.gauge(unit, tm.TM_DOUBLE, tm.TM_RECON_8)
    assert ei.value.status == tm.TM_ERR_PARAM
    # near the singular point the rebuild's error grows like eps / N: the bound is per precision (tm_gauge_load).  A field with one
    # link at N = |U01|^2 + |U02|^2 ~ 1e-6: fp64 takes it (and stays accurate SITE BY SITE, not only in the L2 norm), fp32 / half refuse
    U = np.array(bench.U, copy=True)
    c, s_ = np.cos(7e-4), np.sin(7e-4)
    near = np.array([[c, s_ * 0.6, s_ * 0.8j], [-s_ * 0.6, c, 0], [s_ * 0.8j, 0, c]], dtype=np.complex128)
    near, _ = np.linalg.qr(near)
    near = near * (np.linalg.det(near) ** (-1.0 / 3.0))
    near = near @ np.diag(np.exp(1j * np.array([0.3, -0.1, -0.2])))                 # generic phases, det = 1
    U[2, 37] = near
    n_near = float((np.abs(near[0, 1:]) ** 2).sum())
    assert 1e-8 < n_near < 1e-5
    for prec in (tm.TM_SINGLE, tm.TM_HALF):
        with pytest.raises(tm.TmError) as ei:
            bench.lat.gauge(U, prec, tm.TM_RECON_8)
        assert ei.value.status == tm.TM_ERR_PARAM
    g8 = bench.lat.gauge(U, tm.TM_DOUBLE, tm.TM_RECON_8)
    fin, ftmp, fout = bench.lat.field(tm.TM_DOUBLE, 2).upload(0, psi_e), bench.lat.field(tm.TM_DOUBLE, 2), bench.lat.field(tm.TM_DOUBLE, 2)
    tm.mat_pc(fout, fin, ftmp, g8, pg, tm.TM_MATPC_ASYM, 0)
    bench.lat.sync()
    got, want = fout.download(0), oracle.matpc(psi_e, U, po, oracle.ASYM, 0)
    ev = si.parity_sites(dims, 0)
    site_err = np.abs((got - want)[:, ev]).max(axis=(0, 2, 3)) / np.sqrt((np.abs(want[:, ev]) ** 2).sum(axis=(0, 2, 3)))
    assert site_err.max() <= 1e-9, site_err.max()                                  # eps / N = 1e-16 / 1e-6, with margin


# ---- T7: out-of-bounds stores and races, without compute-sanitizer (closed on this pool: profiles/r2_sanitizer.md) ------------

@pytest.mark.parametrize("variant", VARIANTS, ids=[v[0] for v in VARIANTS])
def test_t7_guard_bands_and_run_to_run_identity(variant):
    """Every kernel type / precision / flavor count of every code path writes into an output field that sits between two 64 KB
    guard bands of a canary pattern (external storage, tm_field_alloc); afterwards the bands are intact (no store outside the
    field, ragged last tile included: 6^4 has 20.25 tiles per parity) and the field is bit-identical to a second and third run
    (the staged kernels read shared memory without a block barrier: a race would show up as a difference between runs)."""
    import torch
    dims = (6, 6, 6, 6)
    bench = bench_for(dims, "haar", 1)
    lat = bench.lat
    tm.tm_set_path(lat.ctx, variant[1])
    for key, val in variant[2].items():
        tm.tm_set_tuning(lat.ctx, key, val)
    GUARD = 64 * 1024
    for kw in (FLAVORS[0], FLAVORS[2]):
        nf = nf_of(kw)
        pg = tm.params(KAPPA, **kw)
        inp, x = si.spinor_field(dims, nf, 2), si.spinor_field(dims, nf, 3)
        for prec in PRECS:
            nbytes = tm.tm_field_bytes(lat.ctx, prec, nf)
            pad = (-nbytes) % 256
            buf = torch.full((GUARD + nbytes + pad + GUARD,), 0xA5, dtype=torch.uint8, device="cuda")
            assert buf.data_ptr() % 256 == 0
            body = buf[GUARD:GUARD + nbytes]
            h = tm.tm_field_alloc(lat.ctx, prec, nf, body.data_ptr(), nbytes)
            try:
                for recon in RECONS + [tm.TM_RECON_8]:
                    g = bench.gauge(prec, recon)
                    for parity, dagger, kt in ((0, 0, 0), (1, 1, 1), (0, 1, 2), (1, 0, 3), (0, 0, 4), (1, 1, 5)):
                        fin = lat.field(prec, nf).upload(1 - parity, si.mask_parity(inp, dims, 1 - parity))
                        fx = lat.field(prec, nf).upload(parity, si.mask_parity(x, dims, parity))
                        runs = []
                        for rep in range(3):
                            body.fill_(0x5A)
                            tm.tm_dslash_apply(h, fin.h, None if kt == 0 else fx.h, g.h, pg, parity, dagger, kt, prec)
                            lat.sync()
                            runs.append(body.clone())
                        assert bool((buf[:GUARD] == 0xA5).all()) and bool((buf[GUARD + nbytes:] == 0xA5).all()), (prec, recon, kt)
                        assert bool((runs[0] == runs[1]).all()) and bool((runs[0] == runs[2]).all()), (prec, recon, kt)
            finally:
                tm.tm_field_free(h)


# ---- T3: composites; BASELINE.json config 1 -------------------------------------------------------

@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
def test_t3_mat_pc_and_reconstruct_match_oracle(kw):
    dims = (4, 4, 4, 8)
    nf = nf_of(kw)
    bench = bench_for(dims, "haar", 1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi = si.spinor_field(dims, nf, 4)
    psi_e, b_o = si.mask_parity(psi, dims, 0), si.mask_parity(si.spinor_field(dims, nf, 6), dims, 1)
    for prec, recon in itertools.product(PRECS, RECONS):
        for typ, dagger in ((tm.TM_MATPC_ASYM, 0), (tm.TM_MATPC_ASYM, 1), (tm.TM_MATPC_SYM, 0)):
            want = oracle.matpc(psi_e, bench.U, po, typ, dagger)
            got = bench.matpc(psi_e, pg, typ, dagger, prec, recon, nf)
            assert rel_l2(got, want) <= TOL[prec], (PREC_NAME[prec], recon, typ, dagger)
        want = oracle.reconstruct_odd(psi_e, b_o, bench.U, po)
        assert rel_l2(bench.reconstruct_odd(psi_e, b_o, pg, prec, recon, nf), want) <= TOL[prec]


def test_t3b_config1_solve_check():
    """BASELINE.json configs[0]: 4^3x8, degenerate, fp64, Haar links seed 1, kappa=0.1632, mu=0.004, antiperiodic.
    Draw a full psi, b = M psi (oracle); the GPU's LHS of Eq. 2.2 applied to psi_e must equal the prepared
    RHS b_e + kappa D_eo R_oo^-1 b_o, and Eq. 2.4 must return psi_o."""
    dims = (4, 4, 4, 8)
    kw = dict(mu=0.004, epsilon=0.0, twist_flavor=1)
    bench = bench_for(dims, "haar", 1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi = si.spinor_field(dims, 1, 1)
    b = oracle.mat(psi, bench.U, po)
    b_e, b_o = si.mask_parity(b, dims, 0), si.mask_parity(b, dims, 1)
    psi_e, psi_o = si.mask_parity(psi, dims, 0), si.mask_parity(psi, dims, 1)
    rhs = b_e + KAPPA * si.mask_parity(oracle.dhop(oracle.twist(b_o, po, inverse=1), bench.U, po), dims, 0)
    for recon in RECONS:
        lhs = bench.matpc(psi_e, pg, tm.TM_MATPC_ASYM, 0, tm.TM_DOUBLE, recon, 1)
        assert rel_l2(lhs, rhs) <= 1e-12
        rec = bench.reconstruct_odd(psi_e, b_o, pg, tm.TM_DOUBLE, recon, 1)
        assert rel_l2(rec, psi_o) <= 1e-12


def test_t3b2_config1_against_the_stored_oracle_samples():
    """The same configs[0] inputs against tests/golden/config1_matpc_asym.txt (oracle outputs stored by a committed
    script that calls only oracle/): sampled components of the LHS of Eq. 2.2 and of Eq. 2.4, fp64, every recon."""
    import os
    dims = (4, 4, 4, 8)
    kw = dict(mu=0.004, epsilon=0.0, twist_flavor=1)
    bench = bench_for(dims, "haar", 1)
    pg = tm.params(KAPPA, **kw)
    psi_e = si.mask_parity(si.spinor_field(dims, 1, 1), dims, 0)
    b_o = si.mask_parity(si.spinor_field(dims, 1, 2), dims, 1)
    rows = [l.split() for l in open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "config1_matpc_asym.txt"))
            if not l.startswith("#")]
    for recon in RECONS + [tm.TM_RECON_8]:
        got = {"matpc_asym": bench.matpc(psi_e, pg, tm.TM_MATPC_ASYM, 0, tm.TM_DOUBLE, recon, 1),
               "reconstruct_odd": bench.reconstruct_odd(psi_e, b_o, pg, tm.TM_DOUBLE, recon, 1)}
        for name, s, sp, c, re, im in rows:
            a = got[name]
            if int(s) < 0:
                assert abs(np.linalg.norm(a.ravel()) - float(re)) <= 1e-12 * float(re)
            else:
                assert abs(a[0, int(s), int(sp), int(c)] - complex(float(re), float(im))) <= 1e-12 * 10


# ---- T3c: the local twist, the twist-free hopping forms, the adjoint of SYM, right-hand sides ----------

@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
def test_t3c_twist_apply_matches_oracle(kw):
    dims = (6, 6, 6, 6)
    nf = nf_of(kw)
    bench = bench_for(dims, "haar", 1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    for parity in (0, 1):
        v = si.mask_parity(si.spinor_field(dims, nf, 21), dims, parity)
        for inverse, dagger in itertools.product((0, 1), (0, 1)):
            want = oracle.twist(v, po, inverse, dagger)
            for prec in PRECS:
                assert rel_l2(bench.twist(v, parity, pg, inverse, dagger, prec, nf), want) <= TOL[prec]
            assert rel_l2(bench.twist(v, parity, pg, inverse, dagger, tm.TM_DOUBLE, nf, in_place=True), want) <= 1e-12


@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
def test_t3d_plain_xpay_axpy_kernels_match_oracle(kw):
    dims = (4, 6, 8, 10)
    nf = nf_of(kw)
    bench = bench_for(dims, "near_identity", 1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    for parity, dagger in itertools.product((0, 1), (0, 1)):
        inp = si.mask_parity(si.spinor_field(dims, nf, 22), dims, 1 - parity)
        x = si.mask_parity(si.spinor_field(dims, nf, 23), dims, parity)
        for kt, coeff in ((tm.TM_DSLASH_XPAY, -KAPPA * KAPPA), (tm.TM_DSLASH_AXPY, KAPPA)):
            want = oracle.hop_xpay(inp, x, bench.U, po, parity, dagger, coeff)
            for prec, recon in itertools.product(PRECS, RECONS):
                got = bench.kernel(inp, x, pg, parity, dagger, kt, prec, recon, nf)
                assert rel_l2(got, want) <= TOL[prec], (PREC_NAME[prec], recon, parity, dagger, kt)


@pytest.mark.parametrize("dims,kind", [((4, 4, 4, 8), "haar"), ((4, 6, 8, 10), "near_identity"), ((6, 6, 6, 6), "haar")])
@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
@pytest.mark.parametrize("path", [0, 1], ids=["packed", "scalar"])
def test_t3g_fused_dslash_twist_inv_kernels_match_oracle(dims, kind, kw, path):
    """The fused D R^-1 kernel types (TM_TWIST_INV_DSLASH_TWIST_INV, TM_RECONSTRUCT_TWIST_INV, TM_DSLASH_TWIST_INV_AXPY: the inverse
    twist applied to the neighbour sites in registers) against oracle.kernel_twist_in: every parity, dagger,
    precision and link compression; the time hops of these kernels read the whole neighbour site."""
    nf = nf_of(kw)
    bench = bench_for(dims, kind, 1)
    tm.tm_set_path(bench.lat.ctx, path)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    full_in, full_x = si.spinor_field(dims, nf, 18), si.spinor_field(dims, nf, 19)
    for parity, dagger, (kt, form) in itertools.product((0, 1), (0, 1), ((tm.TM_TWIST_INV_DSLASH_TWIST_INV, "A"),
                                                                        (tm.TM_RECONSTRUCT_TWIST_INV, "REC"), (tm.TM_DSLASH_TWIST_INV_AXPY, "AXPY"))):
        inp, x = si.mask_parity(full_in, dims, 1 - parity), si.mask_parity(full_x, dims, parity)
        want = oracle.kernel_twist_in(inp, x, bench.U, po, parity, dagger, form)
        for prec, recon in itertools.product(PRECS, RECONS + [tm.TM_RECON_8]):
            got = bench.kernel(inp, None if form == "A" else x, pg, parity, dagger, kt, prec, recon, nf)
            assert "twin" in tm.tm_last_kernel_name(bench.lat.ctx)
            err = rel_l2(got, want)
            assert err <= TOL[prec], (PREC_NAME[prec], recon, parity, dagger, form, err)
            assert np.abs(si.mask_parity(got, dims, 1 - parity)).max() == 0


@pytest.mark.parametrize("kw", FLAVORS, ids=["deg+", "deg-", "ndeg"])
def test_t3e_sym_dagger_is_the_adjoint_and_rhs_preparation(kw):
    dims = (4, 4, 4, 8)
    nf = nf_of(kw)
    bench = bench_for(dims, "haar", 1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    phi = si.mask_parity(si.spinor_field(dims, nf, 24), dims, 0)
    b = si.spinor_field(dims, nf, 25)
    for prec, recon in itertools.product(PRECS, RECONS):
        for typ in (tm.TM_MATPC_ASYM, tm.TM_MATPC_SYM):
            want = oracle.matpc_adjoint(phi, bench.U, po, typ)
            assert rel_l2(bench.matpc(phi, pg, typ, 1, prec, recon, nf), want) <= TOL[prec], (PREC_NAME[prec], recon, typ)
            want = oracle.prepare_rhs(b, bench.U, po, typ)
            assert rel_l2(bench.prepare_rhs(b, pg, typ, prec, recon, nf), want) <= TOL[prec], (PREC_NAME[prec], recon, typ)
        assert rel_l2(bench.prepare_rhs(b, pg, tm.TM_MATPC_SYM, prec, recon, nf, alias=True),
                      oracle.prepare_rhs(b, bench.U, po, tm.TM_MATPC_SYM)) <= TOL[prec]
    # the normal operator M^_sym^dag M^_sym is four launches (the adjoint's leading twist is fused into the D R^-1 kernel) -- five for
    # the half-precision doublet, which keeps the local pass -- and the right-hand side of Eq. 2.2 / 2.3 one launch (two)
    lat = bench.lat
    for prec in PRECS:
        g = bench.gauge(prec, tm.TM_RECON_12)
        f = [lat.field(prec, nf) for _ in range(4)]
        f[0].upload(0, phi)
        n0 = lat.launches()
        tm.mat_pc(f[1], f[0], f[2], g, pg, tm.TM_MATPC_SYM, 0)
        tm.mat_pc(f[3], f[1], f[2], g, pg, tm.TM_MATPC_SYM, 1)
        extra = 1 if (prec == tm.TM_HALF and nf == 2) else 0      # the half doublet keeps the local pass (measured slower fused)
        assert lat.launches() - n0 == 4 + extra
        n0 = lat.launches()
        tm.prepare_rhs(f[3], f[0], f[1], f[2], g, pg, tm.TM_MATPC_SYM)
        assert lat.launches() - n0 == 1 + extra
    lat.sync()


def test_t3f_full_solve_pipeline_on_gpu():
    """b = M psi (oracle, full operator); on the GPU: rhs = tm_prepare_rhs(b), then M^ psi_e == rhs for both
    preconditionings and tm_reconstruct_odd(psi_e, b_o) == psi_o.  fp64, non-degenerate doublet, 4x6x8x10."""
    dims = (4, 6, 8, 10)
    kw = FLAVORS[2]
    bench = bench_for(dims, "near_identity", 1)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi = si.spinor_field(dims, 2, 26)
    b = oracle.mat(psi, bench.U, po)
    psi_e, psi_o = si.mask_parity(psi, dims, 0), si.mask_parity(psi, dims, 1)
    for typ in (tm.TM_MATPC_ASYM, tm.TM_MATPC_SYM):
        rhs = bench.prepare_rhs(b, pg, typ, tm.TM_DOUBLE, tm.TM_RECON_12, 2)
        lhs = bench.matpc(psi_e, pg, typ, 0, tm.TM_DOUBLE, tm.TM_RECON_12, 2)
        assert rel_l2(lhs, rhs) <= 1e-12
    rec = bench.reconstruct_odd(psi_e, si.mask_parity(b, dims, 1), pg, tm.TM_DOUBLE, tm.TM_RECON_12, 2)
    assert rel_l2(rec, psi_o) <= 1e-12


# ---- T4: GPU-side properties that need no oracle --------------------------------------------------

@pytest.mark.parametrize("kw", [FLAVORS[0], FLAVORS[2]], ids=["deg", "ndeg"])
def test_t4_asym_composite_adjointness_on_gpu(kw):
    dims = (8, 8, 8, 8)
    nf = nf_of(kw)
    bench = bench_for(dims, "haar", 11)
    pg = tm.params(KAPPA, **kw)
    psi = si.mask_parity(si.spinor_field(dims, nf, 12), dims, 0)
    phi = si.mask_parity(si.spinor_field(dims, nf, 13), dims, 0)
    for prec, tol in ((tm.TM_DOUBLE, 1e-12), (tm.TM_SINGLE, 1e-5)):
        m_psi = bench.matpc(psi, pg, tm.TM_MATPC_ASYM, 0, prec, tm.TM_RECON_12, nf)
        md_phi = bench.matpc(phi, pg, tm.TM_MATPC_ASYM, 1, prec, tm.TM_RECON_12, nf)
        lhs, rhs = np.vdot(phi, m_psi), np.vdot(md_phi, psi)
        assert abs(lhs - rhs) <= tol * np.linalg.norm(phi) * np.linalg.norm(m_psi)


# ---- T4b: degenerate inputs -----------------------------------------------------------------------------------------

def test_t4b_zero_fields_zero_sites_and_unit_links():
    """The degenerate cases of the method: an all-zero input (half: site norm 0, q 0 -- reading C9), an input that is zero on
    most sites, and the free field (unit links, 18- and 12-real; 8-real refuses them, T2c).  No NaN / inf, exact zeros stay
    zero, and the sparse / free-field results match the oracle."""
    dims = (4, 4, 6, 8)
    lat = tm.Lattice(dims)
    unit = np.zeros((4, lat.V, 3, 3), dtype=np.complex128)
    unit[:, :, [0, 1, 2], [0, 1, 2]] = 1.0
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    sparse = si.mask_parity(si.spinor_field(dims, 2, 81), dims, 0)
    keep = si.parity_sites(dims, 0)[::37]
    mask = np.zeros(lat.V, dtype=bool)
    mask[keep] = True
    sparse[:, ~mask] = 0.0                                   # nonzero on 1 site in 37
    x = si.mask_parity(si.spinor_field(dims, 2, 82), dims, 1)
    for prec, recon in itertools.product(PRECS, RECONS):
        g = lat.gauge(unit, prec, recon)
        zero = lat.field(prec, 2).upload(0, np.zeros_like(sparse))
        fx, fout = lat.field(prec, 2).upload(1, x), lat.field(prec, 2)
        tm.dslash_apply(fout, zero, None, g, pg, 1, 0, 0)                       # A on a zero field
        lat.sync()
        assert np.abs(fout.download(1)).max() == 0.0
        tm.dslash_apply(fout, zero, fx, g, pg, 1, 0, 1)                         # A-xpay: out = x exactly (up to the format)
        lat.sync()
        got = fout.download(1)
        assert np.isfinite(got.view(np.float64)).all()
        assert rel_l2(got, fx.download(1)) <= (0.0 if prec != tm.TM_HALF else 1e-4)
        fin = lat.field(prec, 2).upload(0, sparse)
        for kt in (0, 2):
            tm.dslash_apply(fout, fin, fx, g, pg, 1, 0, kt)
            lat.sync()
            got = fout.download(1)
            assert np.isfinite(got.view(np.float64)).all()
            assert rel_l2(got, oracle.kernel(sparse, x, unit, po, 1, 0, kt)) <= TOL[prec], (PREC_NAME[prec], recon, kt)


# ---- T5: host spin basis (SURVEY.md section 8f "minor": chiral <-> non-relativistic rotation in the pack kernels) ----

def test_t5_host_spin_basis_chiral_and_custom():
    dims = (4, 4, 6, 8)
    bench = bench_for(dims, "haar", 7)
    lat, ctx = bench.lat, bench.lat.ctx
    one = np.eye(2)
    S = np.block([[one, one], [one, -one]]).astype(np.complex128) / np.sqrt(2.0)
    rot = lambda M, a: np.einsum("st,fvtc->fvsc", M, a)
    kw = dict(mu=0.15, epsilon=0.19, twist_flavor=0)
    po, pg = oracle.params(dims, KAPPA, **kw), tm.params(KAPPA, **kw)
    psi_c = si.spinor_field(dims, 2, 61)                       # read as components in the chiral basis
    x_c = si.mask_parity(si.spinor_field(dims, 2, 62), dims, 1)
    try:
        # 1. upload in the chiral basis, download in the kernels' basis: psi_device = S psi_host
        tm.tm_set_host_basis(ctx, tm.TM_BASIS_CHIRAL)
        f = lat.field(tm.TM_DOUBLE, 2).upload(0, psi_c)
        assert rel_l2(f.download(0), si.mask_parity(psi_c, dims, 0)) <= 1e-15       # round trip S^dag S
        tm.tm_set_host_basis(ctx, tm.TM_BASIS_NONREL)
        assert rel_l2(f.download(0), si.mask_parity(rot(S, psi_c), dims, 0)) <= 1e-15
        # 2. gamma5 is diagonal in the chiral basis: (1 + i a gamma5 tau3) multiplies the upper / lower spin halves of
        #    flavor 0 by (1 +- i a) when epsilon = 0 -- a closed form that does not go through S
        kw0 = dict(mu=0.3, epsilon=0.0, twist_flavor=0)
        tm.tm_set_host_basis(ctx, tm.TM_BASIS_CHIRAL)
        fin, fout = lat.field(tm.TM_DOUBLE, 2).upload(0, psi_c), lat.field(tm.TM_DOUBLE, 2)
        tm.twist_apply(fout, fin, tm.params(KAPPA, **kw0), 0, 0)
        got, a = fout.download(0), 2 * KAPPA * 0.3
        want = si.mask_parity(psi_c, dims, 0)
        want[0, :, :2] *= 1 + 1j * a
        want[0, :, 2:] *= 1 - 1j * a
        want[1, :, :2] *= 1 - 1j * a
        want[1, :, 2:] *= 1 + 1j * a
        assert rel_l2(got, want) <= 1e-14
        # 3. every kernel type with chiral host fields = S^dag oracle(S .) in all precisions
        inp_c = si.mask_parity(psi_c, dims, 0)
        for kt, dagger in itertools.product((0, 1, 2, 3), (0, 1)):
            want = rot(S.conj().T, oracle.kernel(rot(S, inp_c), rot(S, x_c), bench.U, po, 1, dagger, kt))
            for prec in PRECS:
                got = bench.kernel(inp_c, None if kt == 0 else x_c, pg, 1, dagger, kt, prec, tm.TM_RECON_12, 2)
                assert rel_l2(got, want) <= TOL[prec], (PREC_NAME[prec], kt, dagger)
        # 4. a custom unitary basis; a non-unitary matrix is refused
        q, _ = np.linalg.qr(np.random.default_rng(5).normal(size=(4, 4)) + 1j * np.random.default_rng(6).normal(size=(4, 4)))
        tm.tm_set_host_basis(ctx, tm.TM_BASIS_CUSTOM, q)
        f = lat.field(tm.TM_DOUBLE, 2).upload(1, psi_c)
        tm.tm_set_host_basis(ctx, tm.TM_BASIS_NONREL)
        assert rel_l2(f.download(1), si.mask_parity(rot(q, psi_c), dims, 1)) <= 1e-15
        with pytest.raises(tm.TmError) as ei:
            tm.tm_set_host_basis(ctx, tm.TM_BASIS_CUSTOM, 1.01 * q)
        assert ei.value.status == tm.TM_ERR_ARG
    finally:
        tm.tm_set_host_basis(ctx, tm.TM_BASIS_NONREL)


# ---- T6: error paths of the boundary --------------------------------------------------------------

def test_t8_launch_timing_modes_pair_and_chained():
    """tm_timing_enable: 1 = an event pair around every launch, 2 = one event between consecutive launches (intervals tile the stream)."""
    import torch
    dims = (16, 16, 16, 16)
    lat = tm.Lattice(dims)
    kw = FLAVORS[0]
    pg = tm.params(KAPPA, **kw)
    g = lat.gauge(si.gauge_field(dims, 5, "haar"), tm.TM_SINGLE, tm.TM_RECON_12)
    f = [lat.field(tm.TM_SINGLE, 1) for _ in range(3)]
    f[0].upload(0, si.mask_parity(si.spinor_field(dims, 1, 6), dims, 0))
    ref = None
    for mode in (1, 2):
        tm.tm_timing_enable(lat.ctx, mode)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(lat.stream)
        for _ in range(10):
            tm.mat_pc(f[1], f[0], f[2], g, pg, tm.TM_MATPC_ASYM, 0)         # two launches
        e1.record(lat.stream)
        rec = tm.tm_timing_read(lat.ctx)
        total = e0.elapsed_time(e1)
        assert len(rec) == 20 and all(ms > 0 for _, ms in rec)
        assert [n for n, _ in rec[:2]] * 10 == [n for n, _ in rec]
        assert sum(ms for _, ms in rec) <= total * 1.001 + 1e-3                # the intervals lie inside the bracket and do not overlap
        assert tm.tm_timing_read(lat.ctx) == []                                # the read clears the log
        tm.mat_pc(f[1], f[0], f[2], g, pg, tm.TM_MATPC_ASYM, 0)             # after a read the chain starts afresh
        assert len(tm.tm_timing_read(lat.ctx)) == 2
        tm.tm_timing_enable(lat.ctx, 0)
        out = f[1].download(0)
        if ref is None:
            ref = out
        assert np.array_equal(out, ref)                                        # timing never changes results
    with pytest.raises(tm.TmError):
        tm.tm_timing_enable(lat.ctx, 3)


@pytest.mark.parametrize("kw", [FLAVORS[0], FLAVORS[2]], ids=["deg+", "ndeg"])
def test_t10_programmatic_dependent_launch_keeps_the_order_of_dependent_kernels(kw):
    """tm_set_tuning("pdl"): the fused kernels are launched with programmatic stream serialization and wait (griddepcontrol.wait) for
    their predecessor before touching a field.  A chain of kernels in which each reads what the previous one wrote, and overwrites what
    the one before that read (RAW and WAR through the same stream), must give bit for bit the results of plain launches -- at a size
    with several waves of blocks (16^3 x 32: 512 blocks of 128 sites, 2048 tiles), in every precision."""
    dims, nf = (16, 16, 16, 32), nf_of(kw)
    lat = tm.Lattice(dims)
    pg = tm.params(KAPPA, **kw)
    U = si.gauge_field(dims, 21, "haar")
    x = si.mask_parity(si.spinor_field(dims, nf, 22), dims, 0)
    for prec in PRECS:
        g = lat.gauge(U, prec, tm.TM_RECON_12)
        f = [lat.field(prec, nf) for _ in range(3)]
        res = {}
        for pdl in (0, 1):
            tm.tm_set_tuning(lat.ctx, "pdl", pdl)
            f[0].upload(0, x)
            for _ in range(6):                       # e -> o -> e -> o ...: f0 -> f1 -> f2 -> f0 -> ... each launch reads the previous output
                tm.dslash_apply(f[1], f[0], None, g, pg, 1, 0, 0)
                tm.dslash_apply(f[2], f[1], f[0], g, pg, 0, 0, 2)
                tm.dslash_apply(f[0], f[2], f[1], g, pg, 1, 1, 1)
            res[pdl] = [f[k].download(p) for k, p in ((0, 1), (1, 1), (2, 0))]
        for a, b in zip(res[0], res[1]):
            assert np.isfinite(a).all() and np.array_equal(a, b), PREC_NAME[prec]
    with pytest.raises(tm.TmError):
        tm.tm_set_tuning(lat.ctx, "pdl", 2)


def test_t9_composites_are_cuda_graph_capturable():
    """The hot path allocates nothing and synchronises nothing once its fields exist: a sequence of tm_mat_pc / tm_dslash_apply calls
    can be captured into a CUDA graph on the context stream and replayed; the replay writes bit for bit what the direct launches wrote."""
    import torch
    dims = (8, 8, 8, 16)
    lat = tm.Lattice(dims)
    s = torch.cuda.Stream()
    lat.use_stream(s)
    sets = []
    for kw in (FLAVORS[0], FLAVORS[2]):
        nf = nf_of(kw)
        pg = tm.params(KAPPA, **kw)
        U = si.gauge_field(dims, 11 + nf, "haar")
        x = si.mask_parity(si.spinor_field(dims, nf, 12 + nf), dims, 0)
        for prec in PRECS:
            g = lat.gauge(U, prec, tm.TM_RECON_12)
            f = [lat.field(prec, nf) for _ in range(4)]
            f[0].upload(0, x)
            sets.append((pg, g, f))

    def step():
        for pg, g, f in sets:
            tm.mat_pc(f[1], f[0], f[2], g, pg, tm.TM_MATPC_ASYM, 0)
            tm.mat_pc(f[3], f[1], f[2], g, pg, tm.TM_MATPC_SYM, 1)
            tm.dslash_apply(f[2], f[3], f[0], g, pg, 1, 0, 1)

    with torch.cuda.stream(s):
        step()                                   # first use: kernels loaded, shared-memory attributes raised
        s.synchronize()
        want = [[f[k].download(1 if k == 2 else 0) for k in (1, 2, 3)] for _, _, f in sets]
        n0 = lat.launches()
        graph = torch.cuda.CUDAGraph()
        graph.capture_begin()
        step()
        graph.capture_end()
        per_step = lat.launches() - n0
        for _, _, f in sets:                     # wipe the outputs, then replay twice
            for k in (1, 2, 3):
                f[k].storage.zero_()
        graph.replay()
        graph.replay()
        s.synchronize()
    assert per_step >= 5 * len(sets) and lat.launches() - n0 == per_step           # a replay launches nothing from the host
    for (_, _, f), w3 in zip(sets, want):
        for k, w in zip((1, 2, 3), w3):
            assert np.array_equal(f[k].download(1 if k == 2 else 0), w)


def test_t6_error_paths():
    dims = (4, 4, 4, 8)
    bench = bench_for(dims, "haar", 1)
    lat = bench.lat
    g = bench.gauge(tm.TM_SINGLE, tm.TM_RECON_12)
    p = tm.params(KAPPA, 0.004)
    a, b, c = lat.field(tm.TM_SINGLE, 1), lat.field(tm.TM_SINGLE, 1), lat.field(tm.TM_SINGLE, 1)
    d64, two = lat.field(tm.TM_DOUBLE, 1), lat.field(tm.TM_SINGLE, 2)

    def status(fn):
        with pytest.raises(tm.TmError) as e:
            fn()
        return e.value.status

    assert status(lambda: tm.dslash_apply(a, a, None, g, p, 0, 0, 0)) == tm.TM_ERR_ALIAS
    assert status(lambda: tm.dslash_apply(a, b, None, g, p, 0, 0, tm.TM_DSLASH_TWIST_XPAY)) == tm.TM_ERR_ARG
    assert status(lambda: tm.dslash_apply(d64, b, None, g, p, 0, 0, 0)) == tm.TM_ERR_MISMATCH
    assert status(lambda: tm.dslash_apply(a, two, None, g, p, 0, 0, 0)) == tm.TM_ERR_MISMATCH
    assert status(lambda: tm.tm_dslash_apply(a.h, b.h, None, g.h, p, 0, 0, 0, tm.TM_DOUBLE)) == tm.TM_ERR_MISMATCH
    assert status(lambda: tm.dslash_apply(a, b, None, g, tm.params(KAPPA, 0.1, twist_flavor=0), 0, 0, 0)) == tm.TM_ERR_MISMATCH
    assert status(lambda: tm.dslash_apply(a, b, None, g, tm.params(KAPPA, 0.1, epsilon=0.1), 0, 0, 0)) == tm.TM_ERR_PARAM
    assert status(lambda: tm.dslash_apply(a, b, None, g, tm.params(KAPPA, 0.1, t_boundary=0), 0, 0, 0)) == tm.TM_ERR_PARAM
    sing = tm.params(KAPPA, 0.0, epsilon=1.0 / (2 * KAPPA), twist_flavor=0)     # 1 + a^2 - b^2 = 0
    t2, t3 = lat.field(tm.TM_SINGLE, 2), lat.field(tm.TM_SINGLE, 2)
    assert status(lambda: tm.dslash_apply(t2, t3, None, g, sing, 0, 0, 0)) == tm.TM_ERR_PARAM
    assert status(lambda: tm.mat_pc(a, a, c, g, p, tm.TM_MATPC_SYM, 1)) == tm.TM_ERR_ALIAS          # out_e is scratch
    assert status(lambda: tm.twist_apply(t2, t3, sing, 1, 0)) == tm.TM_ERR_PARAM
    assert status(lambda: tm.twist_apply(a, t3, p, 0, 0)) == tm.TM_ERR_MISMATCH
    assert status(lambda: tm.dslash_apply(a, b, None, g, p, 0, 0, tm.TM_DSLASH_XPAY)) == tm.TM_ERR_ARG   # needs x
    assert status(lambda: tm.dslash_apply(a, b, c, g, p, 0, 0, 9)) == tm.TM_ERR_ARG
    assert status(lambda: tm.dslash_apply(a, b, None, g, p, 0, 0, tm.TM_RECONSTRUCT_TWIST_INV)) == tm.TM_ERR_ARG   # needs x
    assert status(lambda: tm.prepare_rhs(a, b, c, b, g, p, tm.TM_MATPC_ASYM)) == tm.TM_ERR_ALIAS
    assert status(lambda: tm.mat_pc(a, b, b, g, p, tm.TM_MATPC_ASYM, 0)) == tm.TM_ERR_ALIAS
    assert status(lambda: tm.tm_init((4, 4, 4, 7))) == tm.TM_ERR_DIMS
    assert status(lambda: tm.tm_init((2, 4, 4, 8))) == tm.TM_ERR_DIMS
    # out may alias x (B kernel reads its own site before the store)
    x = si.mask_parity(si.spinor_field(dims, 1, 3), dims, 0)
    inp = si.mask_parity(si.spinor_field(dims, 1, 2), dims, 1)
    fx = lat.field(tm.TM_DOUBLE, 1).upload(0, x)
    fi = lat.field(tm.TM_DOUBLE, 1).upload(1, inp)
    g64 = bench.gauge(tm.TM_DOUBLE, tm.TM_RECON_18)
    tm.dslash_apply(fx, fi, fx, g64, p, 0, 0, tm.TM_DSLASH_TWIST_XPAY)
    lat.sync()
    want = oracle.kernel(inp, x, bench.U, oracle.params(dims, KAPPA, 0.004), 0, 0, oracle.B)
    assert rel_l2(fx.download(0), want) <= 1e-12
    # the launch counter counts dslash kernels
    n0 = lat.launches()
    tm.mat_pc(a, b, c, g, p, tm.TM_MATPC_ASYM, 0)
    assert lat.launches() == n0 + 2
