"""GPU parity of the 16-bit storage path (reading H1): the stored codes are
compared bit for bit with the oracle's, the operator with 16-bit streams against the oracle's
(same storage points), and the reliable-update CG with that operator inside by iteration count
(+-2) and fp64 true residual."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2001_05706_b200 import inputs

from gpu_util import blocks, ctx, pack, parity_mask, relerr, to_dev, unpack

pytestmark = pytest.mark.gpu


def internal_order(c, field_f32, dims):
    """boundary numpy field -> numpy array [2][Vh][24] in the internal (parity, cb) site order."""
    Vh = int(np.prod(dims)) // 2
    p = c.spinor_pack(torch.from_numpy(np.ascontiguousarray(field_f32, dtype=np.float32)).cuda(), dims)
    return p.cpu().numpy().reshape(2, 6, Vh, 4).transpose(0, 2, 1, 3).reshape(2, Vh, 24)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8), (10, 6, 4, 12)])
def test_spinor_codes_and_norms_are_bit_exact(dims):
    c = ctx()
    Vh = int(np.prod(dims)) // 2
    rng = np.random.default_rng(7)
    v = (inputs.spinor_field(dims, 0, 3) * np.exp(rng.uniform(-6, 6, tuple(reversed(dims)) + (1, 1, 1)))).astype(np.float32)
    v[0, 0, 0, 0] = 0.0                                  # an all-zero site
    p32 = c.spinor_pack(torch.from_numpy(v).cuda(), dims)
    half = c.spinor_to_half(p32, dims, 2)
    raw = half.cpu().numpy()
    sites = internal_order(c, v, dims)
    for blk in range(2):
        base = blk * Vh * 52
        codes = raw[base:base + Vh * 48].view(np.int16).reshape(3, Vh, 8).transpose(1, 0, 2).reshape(Vh, 24)
        norms = raw[base + Vh * 48:base + Vh * 52].view(np.float32)
        want_codes, want_norms = orc.q16_codes(sites[blk])
        assert np.array_equal(codes, want_codes)
        assert np.array_equal(norms, want_norms)
    # and the values read back are the oracle's, bit for bit
    back = c.spinor_unpack(c.spinor_from_half(half, dims, 2), dims).cpu().numpy()
    assert np.array_equal(back, orc.q16_spinor(v).reshape(back.shape))


def setup_half(c, dims, kappa, csw):
    U = inputs.gauge_field(dims, 0.5, 0)
    dU = to_dev(U, 8)
    g_hi = c.gauge_load(dU, dims, 8, 18, -1)
    g16 = c.gauge_load(dU, dims, 2, 12, -1)
    A = Ainv = c_hi = c16 = None
    if csw:
        c_hi = c.clover_build(g_hi, kappa, csw, 8)
        c16 = c.clover_build(g_hi, kappa, csw, 2)
        A = orc.clover_matrix(orc.field_strength(U, dims), dims, kappa * csw)
        Ainv = orc.invert_12(A)
    return U, g_hi, g16, c_hi, c16, A, Ainv


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8)])
def test_clover_16bit_storage_matches_oracle(dims):
    c = ctx()
    kappa, csw = 0.135, 1.0
    U, g_hi, g16, c_hi, c16, A, Ainv = setup_half(c, dims, kappa, csw)
    for which, ref in ((0, A), (1, Ainv)):
        got = c.clover_unpack(c16, which).cpu().numpy()
        want = orc.q16_clover(ref).astype(np.float64)
        # codes may differ by one unit where the fp64 -> fp32 rounding of an entry differs in its
        # last bit between the two constructions; one code step is norm/32767
        step = np.abs(want).max(axis=(-3, -2, -1), keepdims=True) / 32767.0
        assert (np.abs(got - want) <= 1.001 * step).all()
        assert (np.abs(got - want) > 1e-9).mean() < 1e-3
        assert relerr(got, want) < 1e-6


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8), (10, 6, 4, 12)])
@pytest.mark.parametrize("csw", [0.0, 1.0])
@pytest.mark.parametrize("dagger", [False, True])
def test_operator_with_16bit_streams_matches_oracle(dims, csw, dagger):
    c = ctx()
    kappa = 0.135
    U, g_hi, g16, c_hi, c16, A, Ainv = setup_half(c, dims, kappa, csw)
    Uq = orc.q16_links(U)
    Aq = None if A is None else orc.q16_clover(A)
    Aiq = None if Ainv is None else orc.q16_clover(Ainv)
    psi = inputs.spinor_field(dims, 0, 2).astype(np.float32)
    psi_q = orc.q16_spinor(psi)
    p32 = c.spinor_pack(torch.from_numpy(psi).cuda(), dims)
    ph = c.spinor_to_half(p32, dims, 2)
    Vh = int(np.prod(dims)) // 2
    flags = 1 if dagger else 0
    # a stored code may flip by one unit (1.5e-5 of the site maximum) where the two fp32
    # evaluation orders round differently: bound the field error well below one code step
    tol = 3e-6
    # full lattice, fp32 output
    out = torch.empty_like(p32)
    c.dslash_half(out, 4, ph, g16, c16, kappa, csw, 2, flags)
    want = orc.apply_M_q16(psi_q, Uq, dims, kappa, Aq, Aiq, -1, 2, dagger, False)
    assert relerr(unpack(c, out, dims), want) <= tol
    # full lattice, 16-bit output
    out16 = c.empty(2 * Vh * 52)
    c.dslash_half(out16, 2, ph, g16, c16, kappa, csw, 2, flags)
    want = orc.apply_M_q16(psi_q, Uq, dims, kappa, Aq, Aiq, -1, 2, dagger, True)
    assert relerr(unpack(c, c.spinor_from_half(out16, dims, 2), dims), want) <= 2e-5
    # even-odd operator on each parity, fp32 output
    m = parity_mask(dims)
    tmp16 = c.empty(Vh * 52)
    for p in (0, 1):
        full = torch.zeros_like(p32)
        c.dslash_half(blocks(full)[p], 4, ph[p * Vh * 52:(p + 1) * Vh * 52], g16, c16, kappa, csw, p, flags, tmp16)
        want = orc.apply_M_q16(psi_q * (m == p), Uq, dims, kappa, Aq, Aiq, -1, p, dagger, False)
        assert relerr(unpack(c, full, dims), want) <= 2e-5


@pytest.mark.parametrize("mode", [2, 0])
def test_half_mixed_cg_matches_oracle(mode):
    """configs[3] at 8^3 x 16 with the 16-bit inner operator."""
    c = ctx()
    dims, kappa, csw, tol = (8, 8, 8, 16), 0.1355, 1.0, 1e-10
    U, g_hi, g16, c_hi, c16, A, Ainv = setup_half(c, dims, kappa, csw)
    b = inputs.spinor_field(dims, 0, 1)
    if mode != 2:
        b = b * (parity_mask(dims) == mode)
    y_ref, st_ref = orc.cg_mixed(b, U, dims, kappa, tol, 5000, A, Ainv, -1, mode, 0.1, half=True)
    c.ensure_workspace(c.workspace_bytes(dims, 8))
    c.set_operator(g_hi, g16, c_hi, c16, kappa, csw, mode, 0.1)
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
    assert st.r_true < 1.5 * tol
    assert relerr(got, y_ref) <= 1e-8


def test_operator_16bit_periodic_t_boundary():
    """t_boundary = +1 (periodic) through the 16-bit kernel: the seam sign is a lane-wise factor of
    the packed arithmetic and must not be folded into the stored links."""
    c = ctx()
    dims, kappa = (6, 4, 2, 8), 0.135
    U = inputs.gauge_field(dims, 0.5, 0)
    g16 = c.gauge_load(to_dev(U, 8), dims, 2, 12, +1)
    Uq = orc.q16_links(U)
    psi = inputs.spinor_field(dims, 0, 5).astype(np.float32)
    psi_q = orc.q16_spinor(psi)
    p32 = c.spinor_pack(torch.from_numpy(psi).cuda(), dims)
    ph = c.spinor_to_half(p32, dims, 2)
    for dagger in (False, True):
        out = torch.empty_like(p32)
        c.dslash_half(out, 4, ph, g16, None, kappa, 0.0, 2, 1 if dagger else 0)
        want = orc.apply_M_q16(psi_q, Uq, dims, kappa, None, None, +1, 2, dagger, False)
        assert relerr(unpack(c, out, dims), want) <= 3e-6
        anti = orc.apply_M_q16(psi_q, Uq, dims, kappa, None, None, -1, 2, dagger, False)
        assert relerr(unpack(c, out, dims), anti) > 1e-3      # and it is not the antiperiodic result
