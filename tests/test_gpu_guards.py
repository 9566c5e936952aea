"""Out-of-bounds writes (compute-sanitizer is closed on this GPU pool): every
output / in-out buffer of the path is a slice of a larger allocation whose guard bands hold a sentinel;
after the call the bands must be untouched.  All field memory is caller-owned, so this covers every
buffer the library may write: hop outputs, the even-odd temporary, 16-bit fields, the multi-rhs batch,
the solver's x and its whole workspace."""
import numpy as np
import pytest
import torch

from paper_2001_05706_b200 import inputs

from gpu_util import ctx, to_dev

pytestmark = pytest.mark.gpu

GUARD = 4096  # elements on each side


class Guarded:
    """n elements of dtype inside sentinel guard bands (the slice start stays 16-byte aligned)"""

    def __init__(self, n, dtype, fill=None):
        self.n, self.dtype = n, dtype
        self.sent = 12345.0 if dtype != torch.uint8 else 0xA5
        self.buf = torch.full((n + 2 * GUARD,), self.sent, dtype=dtype, device="cuda")
        self.t = self.buf[GUARD:GUARD + n]
        if fill is not None:
            self.t.copy_(fill)

    def check(self, what):
        lo, hi = self.buf[:GUARD], self.buf[GUARD + self.n:]
        assert bool((lo == self.sent).all()) and bool((hi == self.sent).all()), "guard band overwritten: " + what


@pytest.mark.parametrize("dims", [(6, 4, 2, 8), (8, 8, 8, 16), (10, 6, 4, 2)])
@pytest.mark.parametrize("precision,recon", [(4, 12), (4, 18), (8, 18)])
def test_operator_outputs_stay_inside_their_buffers(dims, precision, recon):
    c = ctx()
    kappa, csw = 0.135, 1.0
    dt = {4: torch.float32, 8: torch.float64}[precision]
    U = inputs.gauge_field(dims, 0.5, 0)
    g = c.gauge_load(to_dev(U, precision), dims, precision, recon, -1)
    cl = c.clover_build(g, kappa, csw, precision)
    psi = c.spinor_pack(to_dev(inputs.spinor_field(dims, 0, 0), precision), dims)
    h = psi.numel() // 2
    out, tmp, full = Guarded(h, dt), Guarded(h, dt), Guarded(2 * h, dt)
    for dagger in (False, True):
        c.hop(out.t, psi[h:], g, 0, dagger)
        c.hop_xpay(out.t, psi[h:], psi[:h], 1.0, -kappa, g, 0, dagger)
        for p in (0, 1):
            blk = psi[:h] if p == 0 else psi[h:]
            c.dslash_ex(out.t, blk, g, cl, kappa, csw, p, int(dagger), tmp.t)
            c.dslash_ex(out.t, blk, g, None, kappa, 0.0, p, int(dagger), tmp.t)
        c.dslash_ex(full.t, psi, g, cl, kappa, csw, 2, int(dagger), None)
    torch.cuda.synchronize()
    out.check("hop / dslash out"); tmp.check("even-odd temporary"); full.check("full-lattice out")


@pytest.mark.parametrize("dims", [(6, 4, 2, 8), (8, 8, 8, 16)])
def test_half_and_multi_rhs_outputs_stay_inside_their_buffers(dims, monkeypatch):
    c = ctx()
    kappa, csw, nvec = 0.135, 1.0, 5
    U = inputs.gauge_field(dims, 0.5, 0)
    g64 = c.gauge_load(to_dev(U, 8), dims, 8, 18, -1)
    g32 = c.gauge_load(to_dev(U, 8), dims, 4, 12, -1)
    g16 = c.gauge_load(to_dev(U, 8), dims, 2, 12, -1)
    c16 = c.clover_build(g64, kappa, csw, 2)
    psi = c.spinor_pack(to_dev(inputs.spinor_field(dims, 0, 0), 4), dims)
    V = psi.numel() // 24
    hb = (V // 2) * 52
    ph = Guarded(2 * hb, torch.uint8, c.spinor_to_half(psi, dims, 2))
    o16, t16, o32 = Guarded(hb, torch.uint8), Guarded(hb, torch.uint8), Guarded(psi.numel() // 2, torch.float32)
    for flags in (0, 1):
        c.dslash_half(o16.t, 2, ph.t[:hb], g16, c16, kappa, csw, 0, flags, t16.t)
        c.dslash_half(o32.t, 4, ph.t[hb:], g16, None, kappa, 0.0, 1, flags, t16.t)
    batch = torch.cat([psi.roll(i) for i in range(nvec)])
    y = Guarded(batch.numel(), torch.float32)
    ws = Guarded(2 * batch.numel(), torch.float32)
    c.set_workspace(ws.t)
    coeff = inputs.chebyshev_sign_coefficients(6)
    for tile in ("0", "1"):
        monkeypatch.setenv("QCD_MRHS_TILE", tile)
        c.cheb_apply_multi(y.t, batch, nvec, g32, 0.2, coeff, 2.6)
        c.wilson_multi(y.t, batch, nvec, g32, 0.2, True)
    torch.cuda.synchronize()
    c.set_workspace(None)
    for b, what in ((ph, "16-bit input"), (o16, "16-bit out"), (t16, "16-bit temporary"), (o32, "fp32 out of the 16-bit operator"),
                    (y, "multi-rhs out"), (ws, "Chebyshev workspace")):
        b.check(what)


@pytest.mark.parametrize("mode", [0, 2])
@pytest.mark.parametrize("lo", [None, 4, 2])
def test_solvers_stay_inside_x_and_the_workspace(mode, lo):
    c = ctx()
    dims, kappa, csw = (6, 4, 2, 8), 0.135, 1.0
    U = inputs.gauge_field(dims, 0.5, 0)
    g_hi = c.gauge_load(to_dev(U, 8), dims, 8, 18, -1)
    c_hi = c.clover_build(g_hi, kappa, csw, 8)
    g_lo = c.gauge_load(to_dev(U, 8), dims, lo, 12, -1) if lo else None
    c_lo = c.clover_build(g_hi, kappa, csw, lo) if lo else None
    b = c.spinor_pack(to_dev(inputs.spinor_field(dims, 0, 1), 8), dims)
    n = b.numel() if mode == 2 else b.numel() // 2
    x = Guarded(n, torch.float64)
    ws = Guarded(c.workspace_bytes(dims, 8) // 8, torch.float64)
    c.set_workspace(ws.t)
    c.set_operator(g_hi, g_lo, c_hi, c_lo, kappa, csw, mode, 0.1)
    rc, st = c.cg_solve(x.t, b[:n].clone(), 1e-10, 2000)
    assert rc == 0 and st.converged == 1
    if lo is None:
        shifts = [0.0, 0.1, 1.0]
        xs = Guarded(len(shifts) * n, torch.float64)
        wsm = Guarded((4 + len(shifts)) * n, torch.float64)
        c.set_workspace(wsm.t)
        rc, st, _ = c.cg_multishift(xs.t, b[:n].clone(), shifts, 1e-10, 2000)
        assert rc == 0
        torch.cuda.synchronize()
        xs.check("multi-shift x"); wsm.check("multi-shift workspace")
    torch.cuda.synchronize()
    c.set_workspace(None)
    x.check("cg x"); ws.check("cg workspace")
