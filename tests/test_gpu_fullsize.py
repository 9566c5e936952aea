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
