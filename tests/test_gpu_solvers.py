"""GPU parity: fused BLAS, CG on M^dag M, reliable-update mixed CG and the Chebyshev
driver against the CPU oracle (same algorithm, same seeded inputs).  Criteria from
BASELINE.json north_star: iteration count within +-2, true residual below tol."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2001_05706_b200 import inputs, qcd

from gpu_util import TOL, blocks, ctx, pack, parity_mask, relerr, to_dev, unpack

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision", [4, 8])
@pytest.mark.parametrize("n", [4, 24 * 128, 24 * 1000 + 4, 24 * 8 * 8 * 8 * 16])
def test_blas_matches_numpy_fp64(n, precision):
    c = ctx()
    rng = np.random.default_rng(n)
    dt = {4: np.float32, 8: np.float64}[precision]
    x, y, p, q = (rng.standard_normal(n).astype(dt) for _ in range(4))
    X64, Y64, P64, Q64 = (v.astype(np.float64) for v in (x, y, p, q))
    dx, dy, dp, dq = (torch.from_numpy(v).cuda() for v in (x, y, p, q))
    tol = TOL[precision]
    assert abs(c.norm2(dx) - np.dot(X64, X64)) <= 1e-13 * np.dot(X64, X64)
    assert abs(c.redot(dx, dy) - np.dot(X64, Y64)) <= 1e-13 * np.sqrt(np.dot(X64, X64) * np.dot(Y64, Y64))
    # deterministic: same bits every time
    assert c.norm2(dx) == c.norm2(dx)
    a, b = 0.37, -1.21
    t = dy.clone(); c.axpy(a, dx, t)
    assert relerr(t.cpu().numpy(), Y64 + a * X64) <= tol
    t = dy.clone(); c.xpay(dx, a, t)
    assert relerr(t.cpu().numpy(), X64 + a * Y64) <= tol
    t = dy.clone(); c.axpby(a, dx, b, t)
    assert relerr(t.cpu().numpy(), a * X64 + b * Y64) <= tol
    tx, tr = dx.clone(), dy.clone()
    r2 = c.cg_update(a, dp, dq, tx, tr)
    want_r = Y64 - a * Q64
    assert relerr(tx.cpu().numpy(), X64 + a * P64) <= tol
    assert relerr(tr.cpu().numpy(), want_r) <= tol
    got_r = tr.cpu().numpy().astype(np.float64)
    assert abs(r2 - np.dot(got_r, got_r)) <= 1e-13 * r2


def setup_operator(c, dims, kappa, csw, precision, recon, eps=0.5):
    U = inputs.gauge_field(dims, eps, 0)
    if precision == 4:
        U = inputs.round_to_f32(U)
    g = c.gauge_load(to_dev(U, precision), dims, precision, recon, -1)
    A = Ainv = cl = None
    if csw:
        cl = c.clover_build(g, kappa, csw, precision)
        F = orc.field_strength(U, dims)
        A = orc.clover_matrix(F, dims, kappa * csw)
        Ainv = orc.invert_12(A)
    return U, g, cl, A, Ainv


@pytest.mark.parametrize("mode", [2, 0])
@pytest.mark.parametrize("csw,recon", [(0.0, 18), (1.0, 18), (1.0, 12)])
def test_cg_fp64_matches_oracle(mode, csw, recon):
    """configs[2] at a size the oracle finishes in seconds (8^3 x 16; same eps, kappa, csw, tol),
    with 18-real fp64 links and with 12-real ones (row 2 rebuilt in fp64)."""
    c = ctx()
    dims, kappa, tol = (8, 8, 8, 16), 0.135, 1e-10
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, csw, 8, recon)
    b = inputs.spinor_field(dims, 0, 1)
    if mode != 2:
        b = b * (parity_mask(dims) == mode)
    x_ref, st_ref = orc.cg(b, U, dims, kappa, tol, 5000, A, Ainv, -1, mode)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g, None, cl, None, kappa, csw, mode)
    pb = pack(c, b, dims, 8)
    if mode == 2:
        x = torch.empty_like(pb)
        rc, st = c.cg_solve(x, pb, tol, 5000)
        got = unpack(c, x, dims)
    else:
        full = torch.zeros_like(pb)
        rc, st = c.cg_solve(blocks(full)[mode], blocks(pb)[mode], tol, 5000)
        got = unpack(c, full, dims)
    assert rc == 0 and st.converged == 1
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert st.r_true < tol * 1.5 and st.r_iter <= tol
    assert relerr(got, x_ref) <= 1e-8   # both solve N x = b to 1e-10 relative residual; cond(N) ~ 1e2


def test_cg_reports_noconv_and_keeps_iterate():
    c = ctx()
    dims, kappa = (4, 4, 4, 8), 0.135
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, 0.0, 8, 18)
    b = inputs.spinor_field(dims, 0, 1)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g, None, None, None, kappa, 0.0, 2)
    pb = pack(c, b, dims, 8)
    x = torch.empty_like(pb)
    rc, st = c.cg_solve(x, pb, 1e-10, 7)
    assert rc == 1 and st.iters == 7 and st.converged == 0
    x_ref, st_ref = orc.cg(b, U, dims, kappa, 1e-10, 7)
    assert relerr(unpack(c, x, dims), x_ref) <= 1e-11
    assert abs(st.r_true - st_ref["r_true"]) <= 1e-9 * st_ref["r_true"]


def test_cg_zero_source_and_plane_wave():
    """b = 0 -> x = 0 in 0 iterations; free-field plane wave (pin P2) -> 1 iteration."""
    c = ctx()
    dims, kappa = (4, 4, 4, 4), 0.125
    U = inputs.unit_gauge_field(dims)
    g = c.gauge_load(to_dev(U, 8), dims, 8, 12, -1)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g, None, None, None, kappa, 0.0, 2)
    zero = torch.zeros(4 ** 4 * 24, dtype=torch.float64, device="cuda")
    x = torch.ones_like(zero)
    rc, st = c.cg_solve(x, zero, 1e-10, 100)
    assert rc == 0 and st.iters == 0 and float(x.abs().max()) == 0.0
    X, Y, Z, T = dims
    n = (1, 0, 3, 2)
    t, z, y, xx = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    ph = 2 * np.pi * (n[0] * xx / X + n[1] * y / Y + n[2] * z / Z + (n[3] + 0.5) * t / T)
    u = np.random.default_rng(5).standard_normal((4, 3, 2))
    uc = u[..., 0] + 1j * u[..., 1]
    psi = np.exp(1j * ph)[..., None, None] * uc
    b = np.stack([psi.real, psi.imag], axis=-1)
    pb = pack(c, b, dims, 8)
    rc, st = c.cg_solve(x, pb, 1e-10, 100)
    assert rc == 0 and st.iters == 1
    lam = 1.0151650429449555  # SURVEY.md Appendix A.5 (same n, kappa, dims)
    assert relerr(unpack(c, x, dims), b / lam) <= 1e-12


@pytest.mark.parametrize("mode", [2, 0])
def test_mixed_cg_matches_oracle(mode):
    """configs[3] at 8^3 x 16: fp32 12-real inner, fp64 18-real outer, delta = 0.1."""
    c = ctx()
    dims, kappa, csw, tol = (8, 8, 8, 16), 0.1355, 1.0, 1e-10
    U, g_hi, c_hi, A, Ainv = setup_operator(c, dims, kappa, csw, 8, 18)
    g_lo = c.gauge_load(to_dev(U, 8), dims, 4, 12, -1)       # fp64 links rounded to fp32 (S15)
    c_lo = c.clover_build(g_hi, kappa, csw, 4)               # fp64 clover rounded to fp32 (S15)
    b = inputs.spinor_field(dims, 0, 1)
    if mode != 2:
        b = b * (parity_mask(dims) == mode)
    y_ref, st_ref = orc.cg_mixed(b, U, dims, kappa, tol, 5000, A, Ainv, -1, mode, 0.1)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g_hi, g_lo, c_hi, c_lo, kappa, csw, mode, 0.1)
    pb = pack(c, b, dims, 8)
    if mode == 2:
        y = torch.empty_like(pb)
        rc, st = c.cg_solve(y, pb, tol, 5000)
        got = unpack(c, y, dims)
    else:
        full = torch.zeros_like(pb)
        rc, st = c.cg_solve(blocks(full)[mode], blocks(pb)[mode], tol, 5000)
        got = unpack(c, full, dims)
    assert rc == 0 and st.converged == 1
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert abs(st.reliable_updates - st_ref["reliable_updates"]) <= 1
    assert st.r_true < tol * 1.5
    assert relerr(got, y_ref) <= 1e-8


@pytest.mark.parametrize("precision,recon", [(4, 12), (8, 18)])
def test_chebyshev_matches_oracle(precision, recon):
    """configs[4] at 8^3 x 16: degree 100, kappa 0.2, scale 2.6, several vectors."""
    c = ctx()
    dims, kappa, scale = (8, 8, 8, 16), 0.2, 2.6
    U, g, _, _, _ = setup_operator(c, dims, kappa, 0.0, precision, recon)
    coeff = inputs.chebyshev_sign_coefficients(100)
    c.ensure_workspace(c.workspace_bytes(dims, precision))
    for i in range(3):
        v = inputs.spinor_field(dims, 0, 10 + i)
        if precision == 4:
            v = inputs.round_to_f32(v)
        want = orc.cheb(v, U, dims, kappa, coeff, scale)
        pv = pack(c, v, dims, precision)
        y = torch.empty_like(pv)
        c.cheb_apply(y, pv, g, kappa, coeff, scale)
        assert relerr(unpack(c, y, dims), want) <= TOL[precision]
    # low degrees by the same path
    for deg in (0, 1, 2):
        want = orc.cheb(v, U, dims, kappa, coeff[:deg + 1], scale)
        c.cheb_apply(y, pv, g, kappa, coeff[:deg + 1], scale)
        assert relerr(unpack(c, y, dims), want) <= TOL[precision]


@pytest.mark.parametrize("precision,recon,dims", [(4, 12, (8, 8, 8, 16)), (4, 18, (6, 4, 2, 8)), (8, 12, (6, 4, 2, 8)), (8, 18, (4, 4, 4, 4))])
def test_chebyshev_multi_rhs_matches_oracle(precision, recon, dims):
    """nvec right-hand sides per launch, links staged once per block."""
    c = ctx()
    kappa, scale, nvec = 0.2, 2.6, 5
    U, g, _, _, _ = setup_operator(c, dims, kappa, 0.0, precision, recon)
    coeff = inputs.chebyshev_sign_coefficients(40)
    vs = [inputs.spinor_field(dims, 0, 20 + i) for i in range(nvec)]
    if precision == 4:
        vs = [inputs.round_to_f32(v) for v in vs]
    batch = torch.cat([pack(c, v, dims, precision) for v in vs])
    y = torch.empty_like(batch)
    c.ensure_workspace(2 * batch.numel() * batch.element_size())
    c.cheb_apply_multi(y, batch, nvec, g, kappa, coeff, scale)
    n = batch.numel() // nvec
    for i, v in enumerate(vs):
        want = orc.cheb(v, U, dims, kappa, coeff, scale)
        assert relerr(unpack(c, y[i * n:(i + 1) * n].contiguous(), dims), want) <= TOL[precision]
    # the single-vector entry point (links straight from HBM, no staging) agrees with the batch
    y1 = torch.empty_like(batch[:n])
    c.cheb_apply(y1, batch[:n].contiguous(), g, kappa, coeff, scale)
    assert relerr(y1.cpu().numpy(), y[:n].cpu().numpy()) <= (1e-6 if precision == 4 else 1e-14)


@pytest.mark.parametrize("mode,csw,precision,base0", [(2, 0.0, 8, False), (0, 1.0, 8, True), (0, 1.0, 4, True), (2, 1.0, 8, True),
                                                     (0, 1.0, 8, False)])
def test_multishift_cg_matches_oracle(mode, csw, precision, base0):
    """(N + sigma_i) x_i = b for all shifts with one N apply per iteration; base shift 0 (iteration
    fused into the operator's epilogues) and > 0 (separate BLAS kernels), full lattice and even-odd."""
    c = ctx()
    dims, kappa = (8, 8, 8, 16), 0.135
    tol = 1e-10 if precision == 8 else 1e-5
    shifts = [0.0, 0.01, 0.1, 1.0] if base0 else [0.02, 0.3, 3.0]
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, csw, precision, 18)
    if precision == 4 and A is not None:
        A, Ainv = inputs.round_to_f32(A), inputs.round_to_f32(Ainv)
    b = inputs.spinor_field(dims, 0, 1)
    if precision == 4:
        b = inputs.round_to_f32(b)
    if mode != 2:
        b = b * (parity_mask(dims) == mode)
    xs_ref, st_ref = orc.cg_multishift(b, U, dims, kappa, shifts, tol, 5000, A, Ainv, -1, mode)
    pb = pack(c, b, dims, precision)
    n = pb.numel() if mode == 2 else pb.numel() // 2
    src = pb if mode == 2 else blocks(pb)[mode].clone()
    x = torch.empty(len(shifts) * n, dtype=pb.dtype, device="cuda")
    c.ensure_workspace((4 + len(shifts)) * n * precision)
    c.set_operator(g, None, cl, None, kappa, csw, mode)
    rc, st, rts = c.cg_multishift(x, src, shifts, tol, 5000)
    assert rc == 0 and st.converged == 1
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert max(rts) < (1.5 * tol if precision == 8 else 5 * tol)
    for i in range(len(shifts)):
        xi = x[i * n:(i + 1) * n]
        if mode == 2:
            got = unpack(c, xi.contiguous(), dims)
        else:
            full = torch.zeros_like(pb)
            blocks(full)[mode].copy_(xi)
            got = unpack(c, full, dims)
        assert relerr(got, xs_ref[i]) <= (1e-8 if precision == 8 else 1e-3)


def test_multishift_argument_errors():
    from paper_2001_05706_b200 import qcd
    c = ctx()
    dims, kappa = (4, 4, 4, 4), 0.125
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, 0.0, 8, 18)
    c.set_operator(g, None, None, None, kappa, 0.0, 2)
    b = torch.randn(4 ** 4 * 24, device="cuda", dtype=torch.float64)
    x = torch.empty(2 * b.numel(), device="cuda", dtype=torch.float64)
    c.ensure_workspace(6 * b.numel() * 8)
    for bad in ([0.1, 0.1], [0.2, 0.1], [-0.1, 0.1]):
        with pytest.raises(qcd.QcdError) as e:
            c.cg_multishift(x, b, bad, 1e-10, 10)
        assert e.value.code == qcd.EINVAL


# ---- device-side control of the CG drivers ------------------------------
@pytest.mark.parametrize("mixed", [False, True])
def test_cg_run_ahead_does_not_change_the_iteration(mixed, monkeypatch):
    """The host enqueues iterations ahead of the device and the kernels enqueued past the halting
    iteration skip themselves: the result must not depend on how far ahead the host runs
    (QCD_CG_RUNAHEAD = 0 is one poll per iteration) -- same iteration count, same bits."""
    c = ctx()
    dims, kappa, csw, tol = (8, 8, 8, 8), 0.1355, 1.0, 1e-10
    U, g_hi, c_hi, A, Ainv = setup_operator(c, dims, kappa, csw, 8, 18)
    g_lo = c.gauge_load(to_dev(U, 8), dims, 4, 12, -1) if mixed else None
    c_lo = c.clover_build(g_hi, kappa, csw, 4) if mixed else None
    b = inputs.spinor_field(dims, 0, 1) * (parity_mask(dims) == 0)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g_hi, g_lo, c_hi, c_lo, kappa, csw, 0, 0.1)
    pb = pack(c, b, dims, 8)
    res = []
    for ahead in ("0", "1", "2", "7"):
        monkeypatch.setenv("QCD_CG_RUNAHEAD", ahead)
        x = torch.zeros_like(blocks(pb)[0])
        rc, st = c.cg_solve(x, blocks(pb)[0].clone(), tol, 5000)
        assert rc == 0 and st.converged == 1
        res.append((st.iters, st.reliable_updates, st.r_true, x.clone()))
    for it, nup, rt, x in res[1:]:
        assert (it, nup, rt) == res[0][:3]
        assert torch.equal(x, res[0][3])
    if mixed:
        y_ref, st_ref = orc.cg_mixed(b, U, dims, kappa, tol, 5000, A, Ainv, -1, 0, 0.1)
        assert abs(res[0][0] - st_ref["iters"]) <= 2 and abs(res[0][1] - st_ref["reliable_updates"]) <= 1


@pytest.mark.parametrize("mixed", [False, True])
def test_cg_breakdown_leaves_the_iterate_untouched(mixed):
    """<p, N p> = NaN at the first iteration (a NaN in b): QCD_EBREAKDOWN, and the failing update
    has written nothing -- x is still the last iterate (0), not Inf/NaN."""
    from paper_2001_05706_b200 import qcd
    c = ctx()
    dims, kappa, csw = (4, 4, 4, 8), 0.135, 1.0
    U, g_hi, c_hi, A, Ainv = setup_operator(c, dims, kappa, csw, 8, 18)
    g_lo = c.gauge_load(to_dev(U, 8), dims, 4, 12, -1) if mixed else None
    c_lo = c.clover_build(g_hi, kappa, csw, 4) if mixed else None
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g_hi, g_lo, c_hi, c_lo, kappa, csw, 2, 0.1)
    pb = pack(c, inputs.spinor_field(dims, 0, 1), dims, 8)
    pb[17] = float("nan")
    x = torch.full_like(pb, 3.0)
    with pytest.raises(qcd.QcdError) as e:
        c.cg_solve(x, pb, 1e-10, 100)
    assert e.value.code == qcd.EBREAKDOWN
    assert float(x.abs().max()) == 0.0


def test_mixed_cg_maxiter_matches_oracle():
    """maxiter falls between two reliable updates: QCD_NOCONV, iters = maxiter, y = y + x."""
    c = ctx()
    dims, kappa, csw, tol = (4, 4, 4, 8), 0.1355, 1.0, 1e-10
    U, g_hi, c_hi, A, Ainv = setup_operator(c, dims, kappa, csw, 8, 18)
    g_lo = c.gauge_load(to_dev(U, 8), dims, 4, 12, -1)
    c_lo = c.clover_build(g_hi, kappa, csw, 4)
    b = inputs.spinor_field(dims, 0, 1)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g_hi, g_lo, c_hi, c_lo, kappa, csw, 2, 0.1)
    pb = pack(c, b, dims, 8)
    for maxiter in (1, 20, 33):
        y_ref, st_ref = orc.cg_mixed(b, U, dims, kappa, tol, maxiter, A, Ainv, -1, 2, 0.1)
        y = torch.empty_like(pb)
        rc, st = c.cg_solve(y, pb, tol, maxiter)
        assert rc == 1 and st.iters == maxiter == st_ref["iters"]
        assert st.reliable_updates == st_ref["reliable_updates"]
        assert relerr(unpack(c, y, dims), y_ref) <= 1e-5     # fp32 inner iterate
        assert abs(st.r_true - st_ref["r_true"]) <= 1e-3 * st_ref["r_true"]


def test_multishift_cg_long_solve_freezes_converged_shifts():
    """Reading M1 on the GPU: ~470 iterations at kappa = 0.2 with a shift of 10, whose zeta would
    underflow without the freeze (NaN in x_s); every x_s finite and equal to the oracle's."""
    c = ctx()
    dims, kappa, tol = (4, 4, 4, 8), 0.2, 1e-10
    shifts = [0.0, 1.0, 10.0]
    U, g, _, _, _ = setup_operator(c, dims, kappa, 0.0, 8, 18)
    b = inputs.spinor_field(dims, 0, 1)
    xs_ref, st_ref = orc.cg_multishift(b, U, dims, kappa, shifts, tol, 5000)
    pb = pack(c, b, dims, 8)
    n = pb.numel()
    x = torch.empty(len(shifts) * n, dtype=pb.dtype, device="cuda")
    c.ensure_workspace((4 + len(shifts)) * n * 8)
    c.set_operator(g, None, None, None, kappa, 0.0, 2)
    rc, st, rts = c.cg_multishift(x, pb, shifts, tol, 5000)
    assert rc == 0 and st.converged == 1 and st.iters > 300
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert bool(torch.isfinite(x).all())
    assert max(rts) < 1.5 * tol
    for i in range(len(shifts)):
        assert relerr(unpack(c, x[i * n:(i + 1) * n].contiguous(), dims), xs_ref[i]) <= 1e-7


def test_solver_entry_points_reject_wrong_precision_handles():
    """A 16-bit gauge handle where an fp32 / fp64 one is required is QCD_EINVAL, not an
    out-of-bounds read."""
    from paper_2001_05706_b200 import qcd
    c = ctx()
    dims, kappa = (4, 4, 4, 4), 0.125
    U = inputs.gauge_field(dims, 0.5, 0)
    g16 = c.gauge_load(to_dev(U, 8), dims, 2, 12, -1)
    g64 = c.gauge_load(to_dev(U, 8), dims, 8, 18, -1)
    v = torch.randn(4 ** 4 * 24, device="cuda", dtype=torch.float32)
    y = torch.empty_like(v)
    c.ensure_workspace(8 * v.numel() * 8)
    with pytest.raises(qcd.QcdError) as e:
        c.cheb_apply_multi(y, v, 1, g16, kappa, [0.5, 0.25], 2.6)
    assert e.value.code == qcd.EINVAL
    with pytest.raises(qcd.QcdError) as e:
        c.set_operator(g16, None, None, None, kappa, 0.0, 2)
    assert e.value.code == qcd.EINVAL
    with pytest.raises(qcd.QcdError) as e:
        c.set_operator(g64, g64, None, None, kappa, 0.0, 2)       # g_lo must be fp32 or 16-bit
    assert e.value.code == qcd.EINVAL


@pytest.mark.parametrize("dims,variant", [((8, 8, 8, 16), "40"), ((16, 8, 4, 4), "40"), ((16, 8, 4, 4), "41"), ((16, 4, 2, 2), "32")])
def test_chebyshev_multi_rhs_tiled_kernel_matches_oracle(dims, variant, monkeypatch):
    """The opt-in shared-memory tile kernel (hop_tile.cu; north_star (2) "neighbour spinors staged
    through shared memory"): rows of a 4-D tile staged with cp.async, faces read directly.  Both tile
    shapes ((4,4,4,2) for X/2 = 4, (8,4,2,2) for X/2 = 8), tiles that span a whole extent (wrap onto
    themselves), 5 vectors on 4 (3) groups, against the oracle and against the default kernel."""
    c = ctx()
    kappa, scale, nvec = 0.2, 2.6, 5
    U, g, _, _, _ = setup_operator(c, dims, kappa, 0.0, 4, 12)
    coeff = inputs.chebyshev_sign_coefficients(12)
    vs = [inputs.round_to_f32(inputs.spinor_field(dims, 0, 40 + i)) for i in range(nvec)]
    batch = torch.cat([pack(c, v, dims, 4) for v in vs])
    y, y0 = torch.empty_like(batch), torch.empty_like(batch)
    c.ensure_workspace(2 * batch.numel() * 4)
    monkeypatch.setenv("QCD_MRHS_TILE", "0")
    n0 = c.launch_count()
    c.cheb_apply_multi(y0, batch, nvec, g, kappa, coeff, scale)
    monkeypatch.setenv("QCD_MRHS_TILE", "1")
    monkeypatch.setenv("QCD_MRHS_VARIANT", variant)
    c.cheb_apply_multi(y, batch, nvec, g, kappa, coeff, scale)
    n = batch.numel() // nvec
    for i, v in enumerate(vs):
        want = orc.cheb(v, U, dims, kappa, coeff, scale)
        assert relerr(unpack(c, y[i * n:(i + 1) * n].contiguous(), dims), want) <= TOL[4]
    assert relerr(y.cpu().numpy(), y0.cpu().numpy()) <= 1e-6
    out = torch.empty_like(batch)
    c.wilson_multi(out, batch, nvec, g, kappa, True)
    monkeypatch.setenv("QCD_MRHS_TILE", "0")
    out0 = torch.empty_like(batch)
    c.wilson_multi(out0, batch, nvec, g, kappa, True)
    assert relerr(out.cpu().numpy(), out0.cpu().numpy()) <= 1e-6


def test_cg_solve_after_finalize_of_its_ctx_is_an_error_not_a_crash():
    """qcd_cg_solve uses the ctx that last called qcd_set_operator; once that ctx is finalised the call
    must return QCD_EINVAL instead of touching freed memory."""
    import ctypes as C
    from paper_2001_05706_b200 import qcd
    c2 = qcd.Context(0)
    dims, kappa = (4, 4, 4, 4), 0.125
    U = inputs.gauge_field(dims, 0.5, 0)
    g = c2.gauge_load(to_dev(U, 8), dims, 8, 18, -1)
    c2.ensure_workspace(c2.workspace_bytes(dims, 8))
    c2.set_operator(g, None, None, None, kappa, 0.0, 2)
    b = torch.randn(4 ** 4 * 24, device="cuda", dtype=torch.float64)
    x = torch.empty_like(b)
    assert qcd.lib().qcd_cg_solve(C.c_void_p(x.data_ptr()), C.c_void_p(b.data_ptr()), 1e-8, 500) == 0
    torch.cuda.synchronize()
    c2.close()
    rc = qcd.lib().qcd_cg_solve(C.c_void_p(x.data_ptr()), C.c_void_p(b.data_ptr()), 1e-8, 500)
    assert rc == qcd.EINVAL


@pytest.mark.parametrize("dims", [(6, 6, 2, 4), (10, 6, 4, 2), (2, 2, 2, 2)])
@pytest.mark.parametrize("mode", [2, 0, 1])
@pytest.mark.parametrize("mixed", [False, True])
def test_cg_fused_iteration_on_ragged_lattices(dims, mode, mixed):
    """Vh = 144, 240, 8: not multiples of the 64-thread hop block, so the launches that carry the fused
    |t|^2 and the fused residual update run with inactive threads in their last block (they compute a
    clamped site, store nothing and add nothing to the norm).  Against the oracle, all three forms."""
    c = ctx()
    kappa, csw, tol = 0.125, 1.0, 1e-10
    U, g_hi, c_hi, A, Ainv = setup_operator(c, dims, kappa, csw, 8, 18)
    g_lo = c.gauge_load(to_dev(U, 8), dims, 4, 12, -1) if mixed else None
    c_lo = c.clover_build(g_hi, kappa, csw, 4) if mixed else None
    b = inputs.spinor_field(dims, 0, 1)
    if mode != 2:
        b = b * (parity_mask(dims) == mode)
    if mixed:
        x_ref, st_ref = orc.cg_mixed(b, U, dims, kappa, tol, 5000, A, Ainv, -1, mode, 0.1)
    else:
        x_ref, st_ref = orc.cg(b, U, dims, kappa, tol, 5000, A, Ainv, -1, mode)
    c.set_workspace(None)
    c.ensure_workspace(max(c.workspace_bytes(dims, 8), 1 << 16))
    c.set_operator(g_hi, g_lo, c_hi, c_lo, kappa, csw, mode, 0.1)
    pb = pack(c, b, dims, 8)
    if mode == 2:
        x = torch.empty_like(pb)
        rc, st = c.cg_solve(x, pb, tol, 5000)
        got = unpack(c, x, dims)
    else:
        full = torch.zeros_like(pb)
        rc, st = c.cg_solve(blocks(full)[mode], blocks(pb)[mode].clone(), tol, 5000)
        got = unpack(c, full, dims)
    assert rc == 0 and st.converged == 1
    assert abs(st.iters - st_ref["iters"]) <= 2
    assert st.r_true < 1.5 * tol
    assert relerr(got, x_ref) <= 1e-8


@pytest.mark.parametrize("dims", [(8, 8, 8, 16), (6, 4, 2, 8)])
@pytest.mark.parametrize("p", [0, 1])
@pytest.mark.parametrize("csw,precision,recon", [(0.0, 8, 18), (1.0, 8, 18), (1.0, 8, 12), (1.0, 4, 12)])
def test_even_odd_source_preparation_and_reconstruction_match_oracle(dims, p, csw, precision, recon):
    """Reading O5, second half: bhat_p = b_p + kappa H A^-1 b_pb and x_pb = A^-1 (b_pb + kappa H x_p),
    each against the oracle's definition on the same inputs (x_p a random field, not a solution)."""
    c = ctx()
    kappa = 0.135
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, csw, precision, recon)
    b = inputs.spinor_field(dims, 3, 1)
    xp = inputs.spinor_field(dims, 4, 1) * (parity_mask(dims) == p)
    if precision == 4:
        b, xp = inputs.round_to_f32(b), inputs.round_to_f32(xp)
    want_bhat = orc.eo_prepare_source(b, U, dims, kappa, Ainv, -1, p)
    want_x = orc.eo_reconstruct(xp, b, U, dims, kappa, Ainv, -1, p)
    c.ensure_workspace(c.workspace_bytes(dims, precision))
    c.set_operator(g, None, cl, None, kappa, csw, p)
    pb = pack(c, b, dims, precision)
    before = pb.clone()
    full = torch.zeros_like(pb)
    c.eo_prepare(blocks(full)[p], pb)
    assert relerr(unpack(c, full, dims), want_bhat) <= TOL[precision]
    assert torch.equal(blocks(full)[1 - p], torch.zeros_like(blocks(full)[1 - p]))   # only the parity-p block is written
    x = pack(c, xp, dims, precision)
    x_p_before = blocks(x)[p].clone()
    c.eo_reconstruct(x, pb)
    assert torch.equal(blocks(x)[p], x_p_before)
    assert relerr(unpack(c, x, dims), want_x) <= TOL[precision]
    assert torch.equal(pb, before)


@pytest.mark.parametrize("csw", [0.0, 1.0])
def test_full_system_solved_through_the_even_odd_operator(csw):
    """P8 on the GPU: prepare, CG on Mhat^dag Mhat, reconstruct; the result solves (A - kappa H) x = b,
    agrees with the oracle doing the same, and takes the oracle's iteration count +-2."""
    c = ctx()
    dims, kappa, tol = (8, 8, 8, 16), 0.135, 1e-11
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, csw, 8, 18)
    b = inputs.spinor_field(dims, 10, 1)
    bhat = orc.eo_prepare_source(b, U, dims, kappa, Ainv)
    rhs = orc.apply_M(bhat, U, dims, kappa, A, Ainv, mode=0, dagger=True)
    xe, st_ref = orc.cg(rhs, U, dims, kappa, tol, 5000, A, Ainv, -1, 0)
    x_ref = orc.eo_reconstruct(xe, b, U, dims, kappa, Ainv)

    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g, None, cl, None, kappa, csw, 0)
    pb = pack(c, b, dims, 8)
    half = blocks(pb)[0].numel()
    bh = torch.empty(half, dtype=pb.dtype, device="cuda")
    rh = torch.empty_like(bh)
    c.eo_prepare(bh, pb)
    c.apply_operator(rh, bh, qcd.DAGGER)
    x = torch.zeros_like(pb)
    rc, st = c.cg_solve(blocks(x)[0], rh, tol, 5000)
    assert rc == 0 and abs(st.iters - st_ref["iters"]) <= 2
    c.eo_reconstruct(x, pb)
    got = unpack(c, x, dims)
    assert relerr(got, x_ref) <= 1e-9
    Dx = torch.empty_like(pb)
    c.dslash(Dx, x, g, cl, kappa, csw, 2)
    assert relerr(unpack(c, Dx, dims), b) <= 1e-9


@pytest.mark.parametrize("precision", [8, 4])
@pytest.mark.parametrize("inverse", [False, True])
def test_clover_apply_matches_oracle_and_works_in_place(precision, inverse):
    c = ctx()
    dims, kappa, csw = (6, 4, 2, 8), 0.135, 1.0
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, csw, precision, 18)
    v = inputs.spinor_field(dims, 5, 1)
    if precision == 4:
        v = inputs.round_to_f32(v)
    pv = pack(c, v, dims, precision)
    out = torch.zeros_like(pv)
    for p in (0, 1):
        c.clover_apply(blocks(out)[p], blocks(pv)[p], cl, inverse, p)
    want = sum(orc.site_matrix_apply(Ainv if inverse else A, v * (parity_mask(dims) == p), dims, p) for p in (0, 1))
    assert relerr(unpack(c, out, dims), want) <= TOL[precision]
    for p in (0, 1):
        c.clover_apply(blocks(pv)[p], blocks(pv)[p], cl, inverse, p)
    assert torch.equal(pv, out)


def test_even_odd_helpers_argument_errors():
    c = ctx()
    dims, kappa = (4, 4, 4, 4), 0.135
    U, g, cl, A, Ainv = setup_operator(c, dims, kappa, 0.0, 8, 18)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    pb = pack(c, inputs.spinor_field(dims, 0, 1), dims, 8)
    x = torch.zeros_like(pb)
    c.set_operator(g, None, None, None, kappa, 0.0, 2)
    with pytest.raises(qcd.QcdError):
        c.eo_prepare(blocks(x)[0], pb)          # full-lattice operator set
    c.set_operator(g, None, None, None, kappa, 0.0, 0)
    with pytest.raises(qcd.QcdError):
        c.eo_prepare(blocks(pb)[0], pb)         # bhat inside b
    with pytest.raises(qcd.QcdError):
        c.eo_reconstruct(pb, pb)                # x is b


_PDL_SCRIPT = r"""
import hashlib, sys
import numpy as np, torch
from paper_2001_05706_b200 import inputs, qcd
c = qcd.Context(0)
dims, kappa, csw = (8, 8, 8, 8), 0.1355, 1.0
U = inputs.gauge_field(dims, 0.5, 0)
dU = torch.from_numpy(np.ascontiguousarray(U)).cuda()
g_hi = c.gauge_load(dU, dims, 8, 18, -1)
g_lo = c.gauge_load(dU, dims, 4, 12, -1)
g_q = c.gauge_load(dU, dims, 2, 12, -1)
c_hi, c_lo, c_q = (c.clover_build(g_hi, kappa, csw, p) for p in (8, 4, 2))
c.ensure_workspace(c.workspace_bytes(dims, 8))
b = c.spinor_pack(torch.from_numpy(inputs.spinor_field(dims, 0, 1)).cuda(), dims)
h = b.numel() // 2
out = []
for lo, clo in ((None, None), (g_lo, c_lo), (g_q, c_q)):
    c.set_operator(g_hi, lo, c_hi, clo, kappa, csw, 0, 0.1)
    x = torch.zeros_like(b[:h])
    rc, st = c.cg_solve(x, b[:h].clone(), 1e-10, 5000)
    out.append(x)
    print(rc, st.iters, st.reliable_updates)
v = c.spinor_pack(torch.from_numpy(inputs.round_to_f32(inputs.spinor_field(dims, 1, 0))).float().cuda(), dims)
vv = torch.cat([v, 2 * v, -v])
y = torch.empty_like(vv)
c.cheb_apply_multi(y, vv, 3, g_lo, 0.2, [0.3, -0.2, 0.5, 0.1, -0.4], 2.6)
out.append(y)
c.ensure_workspace((4 + 3) * h * 8)
c.set_operator(g_hi, None, c_hi, None, kappa, csw, 0)
xs = torch.empty(3 * h, dtype=b.dtype, device="cuda")
rc, st, rt = c.cg_multishift(xs, b[:h].clone(), [0.0, 0.05, 0.5], 1e-10, 5000)
out.append(xs)
torch.cuda.synchronize()
for t in out:
    print(hashlib.sha256(t.cpu().numpy().tobytes()).hexdigest())
"""


def test_programmatic_dependent_launch_does_not_change_any_result():
    """Every kernel is launched with programmatic stream serialisation by default (QCD_PDL, include/qcd.h) and
    waits on the device for its predecessor before its first read: the solvers (fp64, mixed, 16-bit inside,
    multi-shift) and the multi-rhs Chebyshev driver must give the same bits with it switched off.  The switch is
    read once per process, hence the two child processes."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    outs = []
    for pdl in ("0", "1"):
        env = dict(os.environ, QCD_PDL=pdl, PYTHONPATH=root + os.pathsep + os.environ.get("PYTHONPATH", ""))
        r = subprocess.run([sys.executable, "-c", _PDL_SCRIPT], capture_output=True, text=True, env=env, cwd=root, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout)
    assert outs[0] == outs[1]
    assert len(outs[0].split()) == 9 + 5


def test_repeated_solves_give_the_same_bits():
    """Every reduction is deterministic and every launch waits for its predecessor before its first read
    (programmatic dependent launch): forty repeats of each solver on a lattice small enough for all blocks of
    consecutive launches to be resident together give one result."""
    c = ctx()
    dims, kappa, csw = (8, 8, 8, 8), 0.1355, 1.0
    U, g_hi, c_hi, A, Ainv = setup_operator(c, dims, kappa, csw, 8, 18)
    dU = to_dev(U, 8)
    g_lo, g_q = c.gauge_load(dU, dims, 4, 12, -1), c.gauge_load(dU, dims, 2, 12, -1)
    c_lo, c_q = c.clover_build(g_hi, kappa, csw, 4), c.clover_build(g_hi, kappa, csw, 2)
    pb = pack(c, inputs.spinor_field(dims, 0, 1), dims, 8)
    src = blocks(pb)[0].clone()
    h = src.numel()
    c.ensure_workspace(max(c.workspace_bytes(dims, 8), 7 * h * 8))
    seen = {}
    for _ in range(40):
        for name, lo, clo in (("fp64", None, None), ("mixed", g_lo, c_lo), ("q16", g_q, c_q)):
            c.set_operator(g_hi, lo, c_hi, clo, kappa, csw, 0, 0.1)
            x = torch.zeros_like(src)
            rc, st = c.cg_solve(x, src.clone(), 1e-10, 5000)
            assert rc == 0
            seen.setdefault(name, []).append((st.iters, st.reliable_updates, x))
        c.set_operator(g_hi, None, c_hi, None, kappa, csw, 0)
        xs = torch.empty(3 * h, dtype=src.dtype, device="cuda")
        rc, st, _ = c.cg_multishift(xs, src.clone(), [0.0, 0.05, 0.5], 1e-10, 5000)
        assert rc == 0
        seen.setdefault("multishift", []).append((st.iters, 0, xs))
    for name, runs in seen.items():
        for it, nup, x in runs[1:]:
            assert (it, nup) == runs[0][:2], name
            assert torch.equal(x, runs[0][2]), name
