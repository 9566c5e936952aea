"""GPU parity at BASELINE.json's full size, in the launch configuration bench.py times
(32^3 x 64, fp32, 12-real links, even-odd Wilson-clover operator, kappa 0.1355, csw 1):
the CUDA result is compared with the oracle on SAMPLED output sites the oracle computes one
by one (orc.hop_sites / orc.field_strength_sites), and with properties that hold at any size."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2001_05706_b200 import inputs

from gpu_util import ctx, relerr

pytestmark = pytest.mark.gpu

DIMS = (32, 32, 32, 64)
KAPPA, CSW = 0.1355, 1.0


def assert_every_site_close(got, want, on=None, tol=4e-6):
    """No single site may be off: |got - want|_site <= tol (|want|_site + rms |want|_site).  The rms
    term covers sites whose result is small through cancellation among the 8 hop terms."""
    e = np.linalg.norm((got - want).reshape(-1, 24), axis=1)
    r = np.linalg.norm(want.reshape(-1, 24), axis=1)
    if on is not None:
        e, r = e[on], r[on]
    assert (e <= tol * (r + np.sqrt(np.mean(r * r)))).all(), float((e / (r + np.sqrt(np.mean(r * r)))).max())


def lex(x, y, z, t):
    X, Y, Z, T = DIMS
    return x + X * (y + Y * (z + Z * t))


def neighbours(s):
    X, Y, Z, T = DIMS
    x, y, z, t = s % X, (s // X) % Y, (s // (X * Y)) % Z, s // (X * Y * Z)
    return [lex((x + 1) % X, y, z, t), lex((x - 1) % X, y, z, t), lex(x, (y + 1) % Y, z, t), lex(x, (y - 1) % Y, z, t),
            lex(x, y, (z + 1) % Z, t), lex(x, y, (z - 1) % Z, t), lex(x, y, z, (t + 1) % T), lex(x, y, z, (t - 1) % T)]


def sample_sites(parity, n, seed):
    """corners, seam sites (t = 0, T-1), x-wrap sites and random sites of the given parity."""
    X, Y, Z, T = DIMS
    rng = np.random.default_rng(seed)
    pts = [(0, 0, 0, 0), (X - 1, Y - 1, Z - 1, T - 1), (X - 1, 0, 0, T - 1), (0, Y - 1, Z - 1, 0), (1, 0, 0, 0), (X - 2, 3, 5, T - 1)]
    pts += [tuple(int(v) for v in rng.integers(0, [X, Y, Z, T])) for _ in range(n)]
    out = []
    for (x, y, z, t) in pts:
        if (x + y + z + t) & 1 != parity:
            x = (x + 1) % X
        out.append(lex(x, y, z, t))
    return np.array(sorted(set(out)), dtype=np.int64)


def clover_at(U, sites):
    F = orc.field_strength_sites(U, DIMS, sites)
    A = orc.clover_matrix(F, (len(sites), 1, 1, 1), KAPPA * CSW)
    Ainv = orc.invert_12(A)
    return inputs.round_to_f32(A), inputs.round_to_f32(Ainv)


def site_apply(M, v):
    n = len(v)
    return orc.site_matrix_apply(M, v.reshape(1, 1, 1, n, 4, 3, 2), (n, 1, 1, 1)).reshape(n, 4, 3, 2)


@pytest.fixture(scope="module")
def world():
    c = ctx()
    U = inputs.round_to_f32(inputs.tiled_gauge_field(DIMS, 0.5, 0, 16))
    psi = inputs.round_to_f32(inputs.spinor_field(DIMS, 0, 0))
    dU = torch.from_numpy(U).cuda()
    g = c.gauge_load(dU, DIMS, 4, 12, -1)
    g18 = c.gauge_load(dU, DIMS, 4, 18, -1)
    cl = c.clover_build(g, KAPPA, CSW, 4)
    del dU
    pin = c.spinor_pack(torch.from_numpy(psi).float().cuda(), DIMS)
    return c, U, psi, g, g18, cl, pin


@pytest.mark.parametrize("dagger", [False, True])
def test_hop_sampled_sites_32x64(world, dagger):
    c, U, psi, g, g18, cl, pin = world
    h = pin.numel() // 2
    for gg in (g, g18):
        out = torch.zeros_like(pin)
        c.hop(out[:h], pin[h:], gg, 0, dagger)
        c.hop(out[h:], pin[:h], gg, 1, dagger)
        got = c.spinor_unpack(out, DIMS).cpu().numpy().astype(np.float64).reshape(-1, 4, 3, 2)
        for parity in (0, 1):
            S = sample_sites(parity, 40, 11 + parity)
            want = orc.hop_sites(psi, U, DIMS, S, -1, dagger)
            assert relerr(got[S], want) <= 2e-6
            # per-site too: no sampled site may be off
            err = np.linalg.norm((got[S] - want).reshape(len(S), -1), axis=1) / np.linalg.norm(want.reshape(len(S), -1), axis=1)
            assert err.max() <= 4e-6


@pytest.mark.parametrize("dagger", [False, True])
def test_even_odd_clover_operator_sampled_sites_32x64(world, dagger):
    """The exact call bench.py times: qcd_dslash_ex(parity 0) with the clover handle."""
    c, U, psi, g, g18, cl, pin = world
    h = pin.numel() // 2
    out = torch.zeros_like(pin)
    tmp = torch.empty_like(pin[:h])
    c.dslash_ex(out[:h], pin[:h], g, cl, KAPPA, CSW, 0, 1 if dagger else 0, tmp)
    got = c.spinor_unpack(out, DIMS).cpu().numpy().astype(np.float64).reshape(-1, 4, 3, 2)
    S = sample_sites(0, 24, 5)
    N = np.array(sorted({n for s in S for n in neighbours(int(s))}), dtype=np.int64)
    # psi restricted to the even sites is what the even-odd operator sees
    par = orc.parity_mask_array(DIMS)[..., None, None, None]
    psi_e = psi * (par == 0)
    Hin_N = orc.hop_sites(psi_e, U, DIMS, N, -1, dagger)
    _, Ainv_N = clover_at(U, N)
    t_full = np.zeros_like(psi)
    t_full.reshape(-1, 4, 3, 2)[N] = site_apply(Ainv_N, Hin_N)
    Ht_S = orc.hop_sites(t_full, U, DIMS, S, -1, dagger)
    A_S, _ = clover_at(U, S)
    want = site_apply(A_S, psi.reshape(-1, 4, 3, 2)[S]) - KAPPA ** 2 * Ht_S
    assert relerr(got[S], want) <= 2e-6
    err = np.linalg.norm((got[S] - want).reshape(len(S), -1), axis=1) / np.linalg.norm(want.reshape(len(S), -1), axis=1)
    assert err.max() <= 4e-6
    # odd sites untouched
    assert float(out[h:].abs().max()) == 0.0


@pytest.mark.parametrize("dagger", [False, True])
def test_even_odd_clover_operator_whole_field_32x64(world, dagger):
    """The same call as above, compared with the oracle on EVERY even site (the oracle applies
    Mhat at this size in well under a second once its dense clover field exists)."""
    if _host_mem_gb() < 40:
        pytest.skip("needs ~30 GB of host memory for the oracle's dense clover fields")
    c, U, psi, g, g18, cl, pin = world
    h = pin.numel() // 2
    A = orc.clover_matrix(orc.field_strength(U, DIMS), DIMS, KAPPA * CSW)
    Ainv = inputs.round_to_f32(orc.invert_12(A))
    A = inputs.round_to_f32(A)
    par = orc.parity_mask_array(DIMS)[..., None, None, None]
    tmp = torch.empty_like(pin[:h])
    for p in (0, 1):
        out = torch.zeros_like(pin)
        blk = slice(0, h) if p == 0 else slice(h, 2 * h)
        c.dslash_ex(out[blk], pin[blk], g, cl, KAPPA, CSW, p, 1 if dagger else 0, tmp)
        got = c.spinor_unpack(out, DIMS).cpu().numpy().astype(np.float64)
        want = orc.apply_M(psi * (par == p), U, DIMS, KAPPA, A, Ainv, -1, p, dagger)
        assert relerr(got, want) <= 2e-6
        on = (par == p).ravel()
        assert_every_site_close(got, want, on)
        assert np.abs(got.reshape(-1, 24)[~on]).max() == 0.0        # the other parity is untouched
        del out, got, want


@pytest.mark.parametrize("dagger", [False, True])
def test_hop_whole_field_32x64(world, dagger):
    """Single-parity hop, 12- and 18-real, every site of both parities against the oracle."""
    c, U, psi, g, g18, cl, pin = world
    h = pin.numel() // 2
    want = orc.hop(psi, U, DIMS, -1, dagger)
    for gg in (g, g18):
        out = torch.zeros_like(pin)
        c.hop(out[:h], pin[h:], gg, 0, dagger)
        c.hop(out[h:], pin[:h], gg, 1, dagger)
        got = c.spinor_unpack(out, DIMS).cpu().numpy().astype(np.float64)
        assert relerr(got, want) <= 2e-6
        assert_every_site_close(got, want)
        del out, got


@pytest.mark.parametrize("clover", [False, True])
def test_even_odd_source_preparation_and_reconstruction_whole_field_32x64(world, clover):
    """Reading O5's two ends of an even-odd solve at full size, every site against the oracle's definitions."""
    if clover and _host_mem_gb() < 40:
        pytest.skip("needs ~30 GB of host memory for the oracle's dense clover fields")
    c, U, psi, g, g18, cl, pin = world
    h = pin.numel() // 2
    Ainv = None
    if clover:
        Ainv = inputs.round_to_f32(orc.invert_12(orc.clover_matrix(orc.field_strength(U, DIMS), DIMS, KAPPA * CSW)))
    par = orc.parity_mask_array(DIMS)[..., None, None, None]
    c.ensure_workspace(c.workspace_bytes(DIMS, 4))
    c.set_operator(g, None, cl if clover else None, None, KAPPA, CSW if clover else 0.0, 0)
    out = torch.zeros_like(pin)
    c.eo_prepare(out[:h], pin)
    got = c.spinor_unpack(out, DIMS).cpu().numpy().astype(np.float64)
    want = orc.eo_prepare_source(psi, U, DIMS, KAPPA, Ainv)
    assert relerr(got, want) <= 2e-6
    assert_every_site_close(got, want, (par == 0).ravel())
    # reconstruction from the even block of psi standing in for a solution, b = the prepared field's source
    x = pin.clone()
    x[h:] = 0
    c.eo_reconstruct(x, pin)
    got = c.spinor_unpack(x, DIMS).cpu().numpy().astype(np.float64)
    want = orc.eo_reconstruct(psi * (par == 0), psi, U, DIMS, KAPPA, Ainv)
    assert relerr(got, want) <= 2e-6
    assert_every_site_close(got, want)


def test_operator_adjoint_identity_32x64(world):
    """Re<chi, Mhat psi> = Re<Mhat^dag chi, psi> on the full-size even block (any size property)."""
    c, U, psi, g, g18, cl, pin = world
    h = pin.numel() // 2
    chi = torch.randn(h, device="cuda", dtype=torch.float32, generator=torch.Generator("cuda").manual_seed(3))
    tmp = torch.empty_like(chi)
    Mpsi, Mdchi = torch.empty_like(chi), torch.empty_like(chi)
    src = pin[:h].clone()
    c.dslash_ex(Mpsi, src, g, cl, KAPPA, CSW, 0, 0, tmp)
    c.dslash_ex(Mdchi, chi, g, cl, KAPPA, CSW, 0, 1, tmp)
    lhs, rhs = c.redot(chi, Mpsi), c.redot(Mdchi, src)
    scale = np.sqrt(c.norm2(chi) * c.norm2(Mpsi))
    assert abs(lhs - rhs) <= 2e-6 * scale


# ---- the other configs at their full sizes ------------------------------------------------
def _host_mem_gb():
    try:
        import psutil
        return psutil.virtual_memory().available / 1e9
    except Exception:
        return 0.0


@pytest.mark.parametrize("recon", [18, 12])
@pytest.mark.parametrize("dagger", [False, True])
def test_config1_even_odd_wilson_16x32_fp32_whole_field(recon, dagger):
    """BASELINE.json configs[1] exactly as stated (Table 2 caption for the fp32 /
    12-real setting): 16^3 x 32, fp32, even-odd preconditioned Wilson, eps 0.5, kappa 0.137,
    18- and 12-real link storage; both parities, every site, against the oracle's mode 0 / 1."""
    c = ctx()
    dims, kappa = (16, 16, 16, 32), 0.137
    U = inputs.round_to_f32(inputs.gauge_field(dims, 0.5, 0))
    psi = inputs.round_to_f32(inputs.spinor_field(dims, 0, 0))
    g = c.gauge_load(torch.from_numpy(U).float().cuda(), dims, 4, recon, -1)
    pin = c.spinor_pack(torch.from_numpy(psi).float().cuda(), dims)
    h = pin.numel() // 2
    par = orc.parity_mask_array(dims)[..., None, None, None]
    tmp = torch.empty_like(pin[:h])
    for p in (0, 1):
        out = torch.zeros_like(pin)
        blk = slice(0, h) if p == 0 else slice(h, 2 * h)
        c.dslash_ex(out[blk], pin[blk], g, None, kappa, 0.0, p, 1 if dagger else 0, tmp)
        got = c.spinor_unpack(out, dims).cpu().numpy().astype(np.float64)
        want = orc.apply_M(psi * (par == p), U, dims, kappa, None, None, -1, p, dagger)
        assert relerr(got, want) <= 2e-6
        on = (par == p).ravel()
        assert_every_site_close(got, want, on)
        assert np.abs(got.reshape(-1, 24)[~on]).max() == 0.0


def test_config2_clover_cg_24x64_fp64_full_size():
    """BASELINE.json configs[2] as stated (24^3 x 64, fp64, kappa 0.135, csw 1, tol 1e-10,
    maxiter 5000), even-odd form: iteration count within +-2 of the oracle, true residual
    below tol, solution equal to the oracle's."""
    if _host_mem_gb() < 24:
        pytest.skip("needs ~20 GB of host memory for the oracle's dense clover field")
    c = ctx()
    dims, kappa, csw, tol = (24, 24, 24, 64), 0.135, 1.0, 1e-10
    U = inputs.tiled_gauge_field(dims, 0.5, 0, 16)
    A = orc.clover_matrix(orc.field_strength(U, dims), dims, kappa * csw)
    Ainv = orc.invert_12(A)
    par = orc.parity_mask_array(dims)[..., None, None, None]
    b = inputs.spinor_field(dims, 0, 1) * (par == 0)
    x_ref, st_ref = orc.cg(b, U, dims, kappa, tol, 5000, A, Ainv, -1, 0)
    g = c.gauge_load(torch.from_numpy(U).cuda(), dims, 8, 18, -1)
    cl = c.clover_build(g, kappa, csw, 8)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g, None, cl, None, kappa, csw, 0)
    pb = c.spinor_pack(torch.from_numpy(b).cuda(), dims)
    h = pb.numel() // 2
    full = torch.zeros_like(pb)
    rc, st = c.cg_solve(full[:h], pb[:h], tol, 5000)
    assert rc == 0 and st.converged == 1
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert st.r_true < 1.5 * tol
    assert relerr(c.spinor_unpack(full, dims).cpu().numpy(), x_ref) <= 1e-8


def test_config3_mixed_cg_32x64_full_size(world):
    """BASELINE.json configs[3] as stated (32^3 x 64, fp32 12-real inner / fp64 outer reliable
    updates, kappa 0.1355, csw 1, tol 1e-10), even-odd form, against the oracle's mixed CG."""
    if _host_mem_gb() < 60:
        pytest.skip("needs ~50 GB of host memory for the oracle's dense fp64 + fp32 clover fields")
    c = ctx()
    tol = 1e-10
    U = inputs.tiled_gauge_field(DIMS, 0.5, 0, 16)
    A = orc.clover_matrix(orc.field_strength(U, DIMS), DIMS, KAPPA * CSW)
    Ainv = orc.invert_12(A)
    par = orc.parity_mask_array(DIMS)[..., None, None, None]
    b = inputs.spinor_field(DIMS, 0, 1) * (par == 0)
    y_ref, st_ref = orc.cg_mixed(b, U, DIMS, KAPPA, tol, 5000, A, Ainv, -1, 0, 0.1)
    del A, Ainv
    dU = torch.from_numpy(U).cuda()
    g_hi = c.gauge_load(dU, DIMS, 8, 18, -1)
    g_lo = c.gauge_load(dU, DIMS, 4, 12, -1)
    del dU
    c_hi = c.clover_build(g_hi, KAPPA, CSW, 8)
    c_lo = c.clover_build(g_hi, KAPPA, CSW, 4)
    c.ensure_workspace(c.workspace_bytes(DIMS, 8))
    c.set_operator(g_hi, g_lo, c_hi, c_lo, KAPPA, CSW, 0, 0.1)
    pb = c.spinor_pack(torch.from_numpy(b).cuda(), DIMS)
    h = pb.numel() // 2
    full = torch.zeros_like(pb)
    rc, st = c.cg_solve(full[:h], pb[:h], tol, 5000)
    assert rc == 0 and st.converged == 1
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert abs(st.reliable_updates - st_ref["reliable_updates"]) <= 1
    assert st.r_true < 1.5 * tol
    assert relerr(c.spinor_unpack(full, DIMS).cpu().numpy(), y_ref) <= 1e-8


def test_config4_chebyshev_48x96_reduced_degree_full_size():
    """BASELINE.json configs[4] lattice (48^3 x 96, fp32, 12-real, kappa 0.2): the oracle is too
    slow for degree 100 x 12 vectors at this size, so the full-size check is
    degree 4 on 2 vectors through the multi-rhs entry point, whole field compared."""
    if _host_mem_gb() < 40:
        pytest.skip("needs ~30 GB of host memory")
    c = ctx()
    dims, kappa, scale = (48, 48, 48, 96), 0.2, 2.6
    U = inputs.round_to_f32(inputs.tiled_gauge_field(dims, 0.5, 0, 8))
    coeff = inputs.chebyshev_sign_coefficients(100)[:5]
    g = c.gauge_load(torch.from_numpy(U).float().cuda(), dims, 4, 12, -1)
    vs = [inputs.round_to_f32(inputs.spinor_field(dims, 0, 30 + i)) for i in range(2)]
    batch = torch.cat([c.spinor_pack(torch.from_numpy(v).float().cuda(), dims) for v in vs])
    y = torch.empty_like(batch)
    c.set_workspace(None)
    c.ensure_workspace(2 * batch.numel() * 4)
    c.cheb_apply_multi(y, batch, 2, g, kappa, coeff, scale)
    n = batch.numel() // 2
    for i, v in enumerate(vs):
        want = orc.cheb(v, U, dims, kappa, coeff, scale)
        got = c.spinor_unpack(y[i * n:(i + 1) * n].contiguous(), dims).cpu().numpy()
        assert relerr(got, want) <= 2e-6
    c.set_workspace(None)


# ---- 16-bit storage at full size (reading H1) --------------------------------
def test_half_wilson_full_operator_sampled_sites_32x64(world):
    """D = 1 - kappa H with 16-bit links and a 16-bit input spinor at 32^3 x 64 (full lattice,
    fp32 output), compared on sampled sites with the oracle's hop on the stored-and-read-back
    fields; the stored codes of a sampled site are compared bit for bit."""
    c, U, psi, g, g18, cl, pin = world
    dU = torch.from_numpy(U).cuda()
    g16 = c.gauge_load(dU, DIMS, 2, 12, -1)
    del dU
    Vh = pin.numel() // 48
    ph = c.spinor_to_half(pin, DIMS, 2)
    out = torch.empty_like(pin)
    c.dslash_half(out, 4, ph, g16, None, KAPPA, 0.0, 2, 0)
    got = c.spinor_unpack(out, DIMS).cpu().numpy().astype(np.float64).reshape(-1, 4, 3, 2)
    psi_q = orc.q16_spinor(psi.astype(np.float32)).astype(np.float64)
    back = c.spinor_unpack(c.spinor_from_half(ph, DIMS, 2), DIMS).cpu().numpy()
    assert np.array_equal(back, psi_q.astype(np.float32).reshape(back.shape))
    Uq = orc.q16_links(U.astype(np.float32)).astype(np.float64)
    for parity in (0, 1):
        S = sample_sites(parity, 40, 21 + parity)
        want = psi_q.reshape(-1, 4, 3, 2)[S] - KAPPA * orc.hop_sites(psi_q, Uq, DIMS, S, -1, False)
        assert relerr(got[S], want) <= 2e-6
    del g16


def test_half_mixed_cg_32x64_full_size(world):
    """configs[3] at full size with the 16-bit operator inside the reliable-update CG, against the
    oracle running the same algorithm (half=True): iterations +-2, fp64 true residual below tol."""
    if _host_mem_gb() < 60:
        pytest.skip("needs ~50 GB of host memory for the oracle's dense clover fields")
    c = ctx()
    tol = 1e-10
    U = inputs.tiled_gauge_field(DIMS, 0.5, 0, 16)
    A = orc.clover_matrix(orc.field_strength(U, DIMS), DIMS, KAPPA * CSW)
    Ainv = orc.invert_12(A)
    par = orc.parity_mask_array(DIMS)[..., None, None, None]
    b = inputs.spinor_field(DIMS, 0, 1) * (par == 0)
    y_ref, st_ref = orc.cg_mixed(b, U, DIMS, KAPPA, tol, 5000, A, Ainv, -1, 0, 0.1, half=True)
    del A, Ainv
    dU = torch.from_numpy(U).cuda()
    g_hi = c.gauge_load(dU, DIMS, 8, 18, -1)
    g16 = c.gauge_load(dU, DIMS, 2, 12, -1)
    del dU
    c_hi = c.clover_build(g_hi, KAPPA, CSW, 8)
    c16 = c.clover_build(g_hi, KAPPA, CSW, 2)
    c.ensure_workspace(c.workspace_bytes(DIMS, 8))
    c.set_operator(g_hi, g16, c_hi, c16, KAPPA, CSW, 0, 0.1)
    pb = c.spinor_pack(torch.from_numpy(b).cuda(), DIMS)
    h = pb.numel() // 2
    full = torch.zeros_like(pb)
    rc, st = c.cg_solve(full[:h], pb[:h], tol, 5000)
    assert rc == 0 and st.converged == 1
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert abs(st.reliable_updates - st_ref["reliable_updates"]) <= 1
    assert st.r_true < 1.5 * tol
    assert relerr(c.spinor_unpack(full, DIMS).cpu().numpy(), y_ref) <= 1e-8


# ---- beyond 32-bit byte offsets ----------------------------------------------------------------
def test_hop_64cubed_x64_offsets_beyond_4GB():
    """64^3 x 64 (V = 16.8 M sites): the 18-real gauge field is 4.8 GB in fp32 and 9.7 GB in fp64, so
    the (mu, parity) block offsets and plane strides no longer fit 32 bits.  Sampled sites (the last
    time slices and the mu = 3 links live at the highest addresses) against the oracle."""
    if _host_mem_gb() < 48:
        pytest.skip("needs ~40 GB of host memory")
    c = ctx()
    dims = (64, 64, 64, 64)
    X, Y, Z, T = dims
    U = inputs.round_to_f32(inputs.tiled_gauge_field(dims, 0.5, 0, 8))
    psi = inputs.round_to_f32(inputs.spinor_field(dims, 0, 0))
    dU = torch.from_numpy(U).cuda()
    rng = np.random.default_rng(64)

    def lex64(x, y, z, t):
        return x + X * (y + Y * (z + Z * t))

    pts = [(0, 0, 0, 0), (X - 1, Y - 1, Z - 1, T - 1), (X - 1, 0, Z - 1, T - 1), (0, Y - 1, 0, T - 1), (5, 7, 63, 63), (62, 63, 63, 62)]
    pts += [tuple(int(v) for v in rng.integers(0, [X, Y, Z, T])) for _ in range(40)]
    S = np.array(sorted({lex64(*p) for p in pts}), dtype=np.int64)
    want = orc.hop_sites(psi, U, dims, S, -1, False)
    for precision, tol in ((4, 2e-6), (8, 1e-12)):
        g = c.gauge_load(dU, dims, precision, 18, -1)
        src = torch.from_numpy(psi)
        pin = c.spinor_pack((src.float() if precision == 4 else src).cuda(), dims)
        h = pin.numel() // 2
        out = torch.zeros_like(pin)
        c.hop(out[:h], pin[h:], g, 0, False)
        c.hop(out[h:], pin[:h], g, 1, False)
        got = c.spinor_unpack(out, dims).cpu().numpy().astype(np.float64).reshape(-1, 4, 3, 2)
        assert relerr(got[S], want) <= tol
        err = np.linalg.norm((got[S] - want).reshape(len(S), -1), axis=1) / np.linalg.norm(want.reshape(len(S), -1), axis=1)
        assert err.max() <= 2 * tol
        del g, pin, out, got
        torch.cuda.empty_cache()
