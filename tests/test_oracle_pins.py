"""Pins for the CPU oracle (oracle/): closed forms, invariants, brute force.

The paper prints no equation and no worked numerical example, so the
oracle is pinned by mathematics (SURVEY.md §8(c) pins P1-P11, BASELINE.json
north_star): Clifford algebra, free-field plane waves in closed form,
gamma5-hermiticity, gauge covariance, a constant abelian field (clover
normalisation/sign), a dense 2^4 matrix + LU solve, Schur identities, Chebyshev
identities, and an independently written np.roll-based stencil.
None of these re-type the oracle's site loop.
"""
import os

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2001_05706_b200 import inputs

HERE = os.path.dirname(os.path.abspath(__file__))


def cplx(a):
    return inputs.as_complex(a)


def real(a):
    return inputs.as_real(a)


def vdot(a, b):
    return np.vdot(cplx(a).ravel(), cplx(b).ravel())


def relerr(a, b):
    return np.linalg.norm((np.asarray(a) - np.asarray(b)).ravel()) / np.linalg.norm(np.asarray(b).ravel())


def load_golden_gammas():
    rows = []
    with open(os.path.join(HERE, "golden", "degrand_rossi_gamma.txt")) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            rows.append([complex(*map(float, tok.split(","))) for tok in line.split()])
    return np.array(rows).reshape(4, 4, 4)


# ----------------------------------------------------------------------------- P1
def test_p1_clifford_algebra_and_gamma5():
    g = orc.gamma_matrices()
    for mu in range(4):
        assert np.allclose(g[mu], g[mu].conj().T)                      # Hermitian
        for nu in range(4):
            anti = g[mu] @ g[nu] + g[nu] @ g[mu]
            assert np.allclose(anti, 2.0 * (mu == nu) * np.eye(4))    # {g_mu, g_nu} = 2 delta
        for sgn in (+1, -1):
            P = 0.5 * (np.eye(4) + sgn * g[mu])
            assert np.allclose(P @ P, P)                                # projector
            assert np.linalg.matrix_rank(P) == 2
    assert np.allclose(g[4], g[0] @ g[1] @ g[2] @ g[3])
    assert np.allclose(g[4], np.diag([1, 1, -1, -1]))                  # chiral, diagonal
    assert np.array_equal(g[:4], load_golden_gammas())                 # reading S2 fixture


def test_p1_sigma_block_diagonal_in_chirality():
    g = orc.gamma_matrices()
    s = orc.sigma_matrices()
    planes = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]
    for pl, (m, n) in enumerate(planes):
        assert np.allclose(s[pl], 0.5j * (g[m] @ g[n] - g[n] @ g[m]))
        assert np.allclose(s[pl][:2, 2:], 0) and np.allclose(s[pl][2:, :2], 0)
        assert np.allclose(s[pl], s[pl].conj().T)
    assert np.allclose(s[0], np.diag([1, -1, 1, -1]))                  # sigma_xy
    assert np.allclose(s[5], np.diag([-1, 1, 1, -1]))                  # sigma_zt


# ----------------------------------------------------------------------------- P9
@pytest.mark.parametrize("eps", [0.3, 0.5])
def test_p9_generated_links_are_su3_and_row3_reconstructs(eps):
    U = cplx(inputs.gauge_field((4, 4, 2, 6), eps, seed=3))
    UUd = np.einsum("...ij,...kj->...ik", U, U.conj())
    assert np.abs(UUd - np.eye(3)).max() < 1e-14
    assert np.abs(np.linalg.det(U) - 1).max() < 1e-14
    r3 = np.conj(np.cross(U[..., 0, :], U[..., 1, :]))
    assert np.abs(r3 - U[..., 2, :]).max() < 1e-15
    # not trivially the identity
    assert np.abs(U - np.eye(3)).max() > 0.1


def test_p9_mean_plaquette_matches_recipe():
    # 0.611 (eps=0.3) and 0.239 (eps=0.5) on 8^3x16; smaller lattice, looser bound
    for eps, want in ((0.3, 0.611), (0.5, 0.239)):
        U = cplx(inputs.gauge_field((6, 6, 6, 6), eps, seed=0))
        s = 0.0
        ax = [3, 2, 1, 0]
        for mu in range(4):
            for nu in range(mu + 1, 4):
                Um, Un = U[..., mu, :, :], U[..., nu, :, :]
                P = Um @ np.roll(Un, -1, ax[mu]) @ np.conj(np.swapaxes(np.roll(Um, -1, ax[nu]), -1, -2)) \
                    @ np.conj(np.swapaxes(Un, -1, -2))
                s += np.trace(P, axis1=-2, axis2=-1).real.mean() / 3
        assert abs(s / 6 - want) < 0.02


# ----------------------------------------------------------------------------- P2
def plane_wave(dims, n, u, tb):
    X, Y, Z, T = dims
    p = [2 * np.pi * n[0] / X, 2 * np.pi * n[1] / Y, 2 * np.pi * n[2] / Z,
         2 * np.pi * (n[3] + (0.5 if tb == -1 else 0.0)) / T]
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    phase = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return phase[..., None, None] * u, p


@pytest.mark.parametrize("dims,n,tb", [((4, 4, 4, 4), (1, 0, 3, 2), -1),
                                       ((4, 6, 2, 8), (3, 5, 1, 6), -1),
                                       ((6, 4, 4, 2), (2, 1, 0, 1), +1)])
def test_p2_free_field_plane_wave(dims, n, tb):
    kappa = 0.125
    rng = np.random.default_rng(11)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    psi, p = plane_wave(dims, n, u, tb)
    U = inputs.unit_gauge_field(dims)
    g = load_golden_gammas()
    # D psi = [(1 - 2k sum cos p) + 2ik sum gamma_mu sin p_mu] u e^{ipx}
    Mp = (1 - 2 * kappa * sum(np.cos(p))) * np.eye(4) + 2j * kappa * sum(g[mu] * np.sin(p[mu]) for mu in range(4))
    want = np.einsum("ab,...bc->...ac", Mp, psi)
    got = cplx(orc.apply_M(real(psi), U, dims, kappa, tb=tb))
    assert relerr(got, want) < 1e-13
    # D^dag D psi = lambda psi for ANY u (basis independent scalar)
    lam = (1 - 2 * kappa * sum(np.cos(p))) ** 2 + 4 * kappa ** 2 * sum(np.sin(q) ** 2 for q in p)
    dd = orc.apply_M(orc.apply_M(real(psi), U, dims, kappa, tb=tb), U, dims, kappa, tb=tb, dagger=True)
    assert relerr(cplx(dd), lam * psi) < 1e-13
    # eigenvalues of the 4x4 momentum-space matrix
    ev = np.linalg.eigvals(Mp)
    s2 = np.sqrt(sum(np.sin(q) ** 2 for q in p))
    for sign in (+1, -1):
        assert np.min(np.abs(ev - ((1 - 2 * kappa * sum(np.cos(p))) + sign * 2j * kappa * s2))) < 1e-13


def test_p2_value_from_survey_appendix_a5():
    # 4^4, kappa=0.125, n=(1,0,3,2), antiperiodic t.
    dims, kappa = (4, 4, 4, 4), 0.125
    _, p = plane_wave(dims, (1, 0, 3, 2), np.ones((4, 3)), -1)
    lam = (1 - 2 * kappa * sum(np.cos(p))) ** 2 + 4 * kappa ** 2 * sum(np.sin(q) ** 2 for q in p)
    assert abs(lam - 1.0151650429449555) < 1e-15


def test_p2_cg_on_plane_wave_converges_in_one_iteration():
    dims, kappa, n = (4, 4, 4, 4), 0.125, (1, 0, 3, 2)
    rng = np.random.default_rng(5)
    u = rng.standard_normal((4, 3)) + 1j * rng.standard_normal((4, 3))
    b, p = plane_wave(dims, n, u, -1)
    lam = (1 - 2 * kappa * sum(np.cos(p))) ** 2 + 4 * kappa ** 2 * sum(np.sin(q) ** 2 for q in p)
    x, st = orc.cg(real(b), inputs.unit_gauge_field(dims), dims, kappa, 1e-12, 50)
    assert st["iters"] == 1 and st["converged"]
    assert relerr(cplx(x), b / lam) < 1e-13


# ------------------------------------------------ independent np.roll stencil (brute force)
def roll_hop(psi, U, dims, tb, dagger=False):
    """north_star formula with np.roll shifts; gamma matrices from the fixture."""
    g = load_golden_gammas()
    X, Y, Z, T = dims
    ax = [3, 2, 1, 0]
    out = np.zeros_like(psi)
    sg = -1.0 if dagger else 1.0
    for mu in range(4):
        Um = U[..., mu, :, :]
        fwd = np.roll(psi, -1, ax[mu])                       # psi(x+mu)
        bwd = np.roll(psi, +1, ax[mu])                       # psi(x-mu)
        Ub = np.roll(Um, +1, ax[mu])                         # U_mu(x-mu)
        if mu == 3:
            fwd = fwd.copy(); bwd = bwd.copy()
            fwd[T - 1] *= tb
            bwd[0] *= tb
        cf = np.einsum("...ab,...sb->...sa", Um, fwd)
        cb = np.einsum("...ba,...sb->...sa", Ub.conj(), bwd)
        out += cf - sg * np.einsum("st,...ta->...sa", g[mu], cf)
        out += cb + sg * np.einsum("st,...ta->...sa", g[mu], cb)
    return out


@pytest.mark.parametrize("dims", [(4, 6, 2, 8), (2, 2, 2, 2), (6, 2, 4, 4)])
@pytest.mark.parametrize("dagger", [False, True])
def test_hop_matches_roll_stencil(dims, dagger):
    U = inputs.gauge_field(dims, 0.5, seed=1)
    psi = inputs.spinor_field(dims, seed=1)
    got = cplx(orc.hop(psi, U, dims, tb=-1, dagger=dagger))
    want = roll_hop(cplx(psi), cplx(U), dims, -1, dagger)
    assert relerr(got, want) < 1e-14
    # parity-masked form: same values on that parity, zero elsewhere
    par = orc.parity_mask_array(dims)
    for p in (0, 1):
        gp = cplx(orc.hop(psi, U, dims, tb=-1, dagger=dagger, parity_mask=p))
        assert np.array_equal(gp[par == p], got[par == p])
        assert np.all(gp[par != p] == 0)
    # sampled evaluation agrees with the full one
    V = int(np.prod(dims))
    sites = np.array([0, 1, V // 3, V - 1])
    gs = cplx(orc.hop_sites(psi, U, dims, sites, tb=-1, dagger=dagger))
    assert np.array_equal(gs, got.reshape(V, 4, 3)[sites])


def test_hop_is_parity_odd():
    dims = (4, 4, 2, 6)
    U = inputs.gauge_field(dims, 0.5, seed=2)
    psi = inputs.spinor_field(dims, seed=2)
    par = orc.parity_mask_array(dims)
    psi_e = psi * (par == 0)[..., None, None, None]
    h = orc.hop(psi_e, U, dims)
    assert np.all(h[par == 0] == 0) and np.abs(h[par == 1]).max() > 0


# ----------------------------------------------------------------------------- clover helpers
def clover_fields(U, dims, kappa, csw):
    F = orc.field_strength(U, dims)
    A = orc.clover_matrix(F, dims, kappa * csw)
    return F, A, orc.invert_12(A)


# ----------------------------------------------------------------------------- P3
@pytest.mark.parametrize("clover", [False, True])
def test_p3_gamma5_hermiticity(clover):
    dims, kappa = (4, 4, 2, 6), 0.135
    U = inputs.gauge_field(dims, 0.5, seed=4)
    A = Ainv = None
    if clover:
        _, A, Ainv = clover_fields(U, dims, kappa, 1.0)
    chi, psi = inputs.spinor_field(dims, 4, 0), inputs.spinor_field(dims, 4, 1)
    g5 = np.array([1, 1, -1, -1.0])[:, None, None]
    for mode in (2, 0, 1):
        if mode != 2:
            par = orc.parity_mask_array(dims)
            m = (par == mode)[..., None, None, None]
            c, p = chi * m, psi * m
        else:
            c, p = chi, psi
        lhs = vdot(c, g5 * orc.apply_M(p, U, dims, kappa, A, Ainv, mode=mode))
        rhs = vdot(g5 * orc.apply_M(c, U, dims, kappa, A, Ainv, mode=mode), p)
        assert abs(lhs - rhs) < 1e-11 * abs(lhs)
        # explicit adjoint == gamma5 M gamma5, and <chi, M psi> = <M^dag chi, psi>
        Md = orc.apply_M(c, U, dims, kappa, A, Ainv, mode=mode, dagger=True)
        assert relerr(Md, g5 * orc.apply_M(g5 * c, U, dims, kappa, A, Ainv, mode=mode)) < 1e-13
        assert abs(vdot(c, orc.apply_M(p, U, dims, kappa, A, Ainv, mode=mode)) - vdot(Md, p)) < 1e-11 * abs(lhs)


# ----------------------------------------------------------------------------- P4
def gauge_transform(U, g, dims):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag."""
    ax = [3, 2, 1, 0]
    Uc = cplx(U)
    out = np.empty_like(Uc)
    for mu in range(4):
        gp = np.roll(g, -1, ax[mu])
        out[..., mu, :, :] = g @ Uc[..., mu, :, :] @ np.conj(np.swapaxes(gp, -1, -2))
    return real(out)


@pytest.mark.parametrize("clover", [False, True])
def test_p4_gauge_covariance(clover):
    dims, kappa = (4, 2, 6, 4), 0.135
    U = inputs.gauge_field(dims, 0.5, seed=6)
    g = inputs.su3_site_field(dims, 1.0, seed=6)
    psi = inputs.spinor_field(dims, 6)
    U2 = gauge_transform(U, g, dims)
    psi2 = real(np.einsum("...ab,...sb->...sa", g, cplx(psi)))
    A = A2 = None
    if clover:
        _, A, _ = clover_fields(U, dims, kappa, 1.0)
        _, A2, _ = clover_fields(U2, dims, kappa, 1.0)
    lhs = cplx(orc.apply_M(psi2, U2, dims, kappa, A2))
    rhs = np.einsum("...ab,...sb->...sa", g, cplx(orc.apply_M(psi, U, dims, kappa, A)))
    assert relerr(lhs, rhs) < 1e-13
    if clover:   # F transforms in the adjoint: F'(x) = g F g^dag
        F = cplx(orc.field_strength(U, dims)); F2 = cplx(orc.field_strength(U2, dims))
        gF = g[..., None, :, :] @ F @ np.conj(np.swapaxes(g, -1, -2))[..., None, :, :]
        assert relerr(F2, gF) < 1e-13


# ----------------------------------------------------------------------------- P6 / P7
PLANES = [(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)]


def abelian_field(dims, m, n, k=1):
    """Constant abelian field in the (m, n) plane, m < n (SURVEY.md 8(c) P6 rotated into every plane):
    U_m(x) = exp(-i B x_n Tg), U_n(x) = exp(+i B L_n x_m Tg) on x_n = L_n - 1 (else 1), all other links 1,
    Tg = diag(1,-1,0), B = 2 pi k / (L_m L_n).  Every mn-plaquette U_m(x) U_n(x+m) U_m(x+n)^+ U_n(x)^+
    equals exp(i B Tg), also across the x_n seam (B L_m L_n = 2 pi k); every other plaquette is 1."""
    X, Y, Z, T = dims
    B = 2 * np.pi * k / (dims[m] * dims[n])
    Tg = np.array([1.0, -1.0, 0.0])
    U = np.zeros((T, Z, Y, X, 4, 3, 3), dtype=complex)
    for a in range(3):
        U[..., :, a, a] = 1.0
    coord = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")[::-1]  # x, y, z, t
    xm, xn = coord[m], coord[n]
    for a in range(3):
        U[..., m, a, a] = np.exp(-1j * B * xn * Tg[a])
        U[..., n, a, a] = np.where(xn == dims[n] - 1, np.exp(1j * B * dims[n] * xm * Tg[a]), 1.0)
    return U, B, Tg


@pytest.mark.parametrize("plane", range(6))
def test_p6_constant_abelian_field_pins_clover_in_every_plane(plane):
    # Fhat_mn = i sin(B Tg) in the plane that carries the field, 0 in the other five, and
    # C = - sigma_mn (x) sin(B Tg) with sigma_mn = (i/2)[g_m, g_n] from the golden gamma fixture:
    # pins the 1/8, the four leaves, the orientation and the i sigma sign plane by plane.
    m, n = PLANES[plane]
    dims = (4, 6, 4, 2) if plane == 0 else (4, 6, 2, 4)
    U, B, Tg = abelian_field(dims, m, n)
    # the construction itself: plaquettes by np.roll, independent of the oracle
    ax = [3, 2, 1, 0]
    dag = lambda M: np.conj(np.swapaxes(M, -1, -2))
    for (a, b) in PLANES:
        Ua, Ub = U[..., a, :, :], U[..., b, :, :]
        P = Ua @ np.roll(Ub, -1, ax[a]) @ dag(np.roll(Ua, -1, ax[b])) @ dag(Ub)
        want = np.diag(np.exp(1j * B * Tg)) if (a, b) == (m, n) else np.eye(3)
        assert np.abs(P - want).max() < 1e-14
    F = cplx(orc.field_strength(real(U), dims))
    for pl in range(6):
        want = np.diag(1j * np.sin(B * Tg)) if pl == plane else np.zeros((3, 3))
        assert np.abs(F[..., pl, :, :] - want).max() < 1e-15, (plane, pl)
    g = load_golden_gammas()
    sigma = 0.5j * (g[m] @ g[n] - g[n] @ g[m])
    C = cplx(orc.clover_matrix(real(F), dims, 1.0, add_unit=False))
    want = -np.kron(sigma, np.diag(np.sin(B * Tg)))
    assert np.abs(C - want).max() < 1e-15
    assert np.abs(want).max() > 0.2
    # and with the coefficient and the unit matrix: A = 1 + kappa csw C
    A = cplx(orc.clover_matrix(real(F), dims, 0.135 * 1.7))
    assert np.abs(A - (np.eye(12) + 0.135 * 1.7 * want)).max() < 1e-15


def test_p6_abelian_fields_in_two_planes_superpose():
    # fields in the xy and the zt plane at once (they commute): F_xy and F_zt both i sin(B Tg),
    # with different B, the other four planes 0 -- a per-plane sign or index slip cannot hide
    dims = (4, 6, 4, 2)
    U1, B1, Tg = abelian_field(dims, 0, 1)
    U2, B2, _ = abelian_field(dims, 2, 3)
    U = U1 @ U2                                      # link by link; diagonal, so the order is immaterial
    F = cplx(orc.field_strength(real(U), dims))
    for pl in range(6):
        want = {0: np.diag(1j * np.sin(B1 * Tg)), 5: np.diag(1j * np.sin(B2 * Tg))}.get(pl, np.zeros((3, 3)))
        assert np.abs(F[..., pl, :, :] - want).max() < 1e-15, pl
    assert abs(B1 - B2) > 0.1


def test_p7_clover_structure_and_inverse():
    dims, kappa, csw = (4, 4, 4, 2), 0.135, 1.0
    U = inputs.gauge_field(dims, 0.5, seed=8)
    F, A, Ainv = clover_fields(U, dims, kappa, csw)
    Fc = cplx(F)
    assert np.abs(Fc + np.conj(np.swapaxes(Fc, -1, -2))).max() < 1e-15      # anti-Hermitian
    C = cplx(orc.clover_matrix(F, dims, 1.0, add_unit=False))
    assert np.abs(C - np.conj(np.swapaxes(C, -1, -2))).max() < 1e-15       # Hermitian
    assert np.abs(np.trace(C, axis1=-2, axis2=-1)).max() < 1e-14           # traceless
    assert np.abs(C[..., :6, 6:]).max() == 0 and np.abs(C[..., 6:, :6]).max() == 0
    Ac, Ai = cplx(A), cplx(Ainv)
    assert np.abs(Ac - (np.eye(12) + kappa * csw * C)).max() < 1e-15
    assert np.abs(Ac @ Ai - np.eye(12)).max() < 1e-13
    assert np.abs(Ai - np.linalg.inv(Ac)).max() < 1e-13                    # library routine
    ev = np.linalg.eigvalsh(Ac)
    assert ev.min() > 0.5 and ev.max() < 1.5
    # sampled evaluation
    V = int(np.prod(dims)); sites = np.array([0, 7, V - 1])
    Fs = orc.field_strength_sites(U, dims, sites)
    assert np.array_equal(Fs, F.reshape(V, 6, 3, 3, 2)[sites])


# ----------------------------------------------------------------------------- P5
def dense_matrix(apply, dims):
    V = int(np.prod(dims)); n = 12 * V
    D = np.zeros((n, n), dtype=complex)
    e = np.zeros(n, dtype=complex)
    shape = (dims[3], dims[2], dims[1], dims[0], 4, 3)
    for j in range(n):
        e[:] = 0; e[j] = 1
        D[:, j] = cplx(apply(real(e.reshape(shape)))).ravel()
    return D


@pytest.mark.parametrize("clover", [False, True])
def test_p5_dense_2to4_matrix_and_cg(clover):
    dims, kappa = (2, 2, 2, 2), 0.135
    U = inputs.gauge_field(dims, 0.5, seed=9)
    A = Ainv = None
    if clover:
        _, A, Ainv = clover_fields(U, dims, kappa, 1.0)
    D = dense_matrix(lambda v: orc.apply_M(v, U, dims, kappa, A), dims)
    Dd = dense_matrix(lambda v: orc.apply_M(v, U, dims, kappa, A, dagger=True), dims)
    assert np.abs(Dd - D.conj().T).max() < 1e-14                         # explicit adjoint
    G5 = np.kron(np.eye(16), np.kron(np.diag([1, 1, -1, -1.0]), np.eye(3)))
    assert np.abs(G5 @ D @ G5 - D.conj().T).max() < 1e-14               # gamma5 hermiticity, entrywise
    b = inputs.spinor_field(dims, 9)
    N = D.conj().T @ D
    xs = np.linalg.solve(N, cplx(b).ravel())
    x, st = orc.cg(b, U, dims, kappa, 1e-12, 1000, A=A)
    assert st["converged"] and st["r_true"] < 2e-12
    assert relerr(cplx(x).ravel(), xs) < 1e-10
    # CG cannot need more iterations than the dimension; and is not trivially short
    assert 20 < st["iters"] <= 192
    # even-odd operator against the dense Schur complement
    par = orc.parity_mask_array(dims).ravel()
    idx = lambda p: np.repeat(par == p, 12)
    Dee, Deo = D[np.ix_(idx(0), idx(0))], D[np.ix_(idx(0), idx(1))]
    Doe, Doo = D[np.ix_(idx(1), idx(0))], D[np.ix_(idx(1), idx(1))]
    S = Dee - Deo @ np.linalg.inv(Doo) @ Doe
    Mh = dense_matrix(lambda v: orc.apply_M(v * (orc.parity_mask_array(dims) == 0)[..., None, None, None],
                                            U, dims, kappa, A, Ainv, mode=0), dims)
    assert np.abs(Mh[np.ix_(idx(0), idx(0))] - S).max() < 1e-13
    assert np.abs(Mh[np.ix_(idx(1), idx(0))]).max() == 0


# ----------------------------------------------------------------------------- P8
@pytest.mark.parametrize("clover", [False, True])
def test_p8_schur_solve_reconstructs_full_solution(clover):
    dims, kappa = (4, 4, 4, 8), 0.135
    U = inputs.gauge_field(dims, 0.5, seed=10)
    A = Ainv = None
    if clover:
        _, A, Ainv = clover_fields(U, dims, kappa, 1.0)
    b = inputs.spinor_field(dims, 10)
    # solve D x = b through the even-odd system: Mhat x_e = bhat_e via CG on Mhat^dag Mhat
    bhat = orc.eo_prepare_source(b, U, dims, kappa, Ainv)
    rhs = orc.apply_M(bhat, U, dims, kappa, A, Ainv, mode=0, dagger=True)
    xe, st = orc.cg(rhs, U, dims, kappa, 1e-12, 2000, A=A, Ainv=Ainv, mode=0)
    assert st["converged"]
    x = orc.eo_reconstruct(xe, b, U, dims, kappa, Ainv)
    assert relerr(orc.apply_M(x, U, dims, kappa, A), b) < 1e-10
    # even-odd CG needs far fewer iterations than the full-lattice one (134 vs 56)
    rhs_full = orc.apply_M(b, U, dims, kappa, A, dagger=True)
    _, stf = orc.cg(rhs_full, U, dims, kappa, 1e-12, 2000, A=A)
    assert st["iters"] < 0.7 * stf["iters"]


# ----------------------------------------------------------------------------- P10
def test_p10_chebyshev_recurrence():
    dims, kappa, scale = (4, 4, 4, 4), 0.2, 2.6
    U = inputs.gauge_field(dims, 0.5, seed=12)
    v = inputs.spinor_field(dims, 12)
    X = lambda w: orc.apply_HW(w, U, dims, kappa) / scale
    # H_W = gamma5 (1 - kappa H) is Hermitian
    w = inputs.spinor_field(dims, 12, 1)
    assert abs(vdot(w, X(v)) - vdot(X(w), v)) < 1e-12 * abs(vdot(w, X(v)))
    # degree 0, 1, 2 by hand
    c = np.array([0.3, -1.1, 0.7])
    assert relerr(orc.cheb(v, U, dims, kappa, c[:1], scale), c[0] * v) < 1e-15
    assert relerr(orc.cheb(v, U, dims, kappa, c[:2], scale), c[0] * v + c[1] * X(v)) < 1e-15
    t2 = 2 * X(X(v)) - v
    assert relerr(orc.cheb(v, U, dims, kappa, c, scale), c[0] * v + c[1] * X(v) + c[2] * t2) < 1e-15
    # forward recurrence == Clenshaw (different evaluation order), degree 40
    coeff = inputs.chebyshev_sign_coefficients(40, 0.01)
    y = orc.cheb(v, U, dims, kappa, coeff, scale)
    b1 = np.zeros_like(v); b2 = np.zeros_like(v)
    for k in range(len(coeff) - 1, 0, -1):
        b1, b2 = coeff[k] * v + 2 * X(b1) - b2, b1
    yc = coeff[0] * v + X(b1) - b2
    assert relerr(y, yc) < 1e-14


def test_p10_chebyshev_on_free_field_eigenvector_is_scalar_polynomial():
    dims, kappa, scale, tb = (4, 4, 4, 4), 0.2, 2.6, -1
    g = load_golden_gammas()
    _, p = plane_wave(dims, (1, 0, 3, 2), np.ones((4, 3)), tb)
    Mp = (1 - 2 * kappa * sum(np.cos(p))) * np.eye(4) + 2j * kappa * sum(g[mu] * np.sin(p[mu]) for mu in range(4))
    Hp = np.diag([1, 1, -1, -1.0]) @ Mp
    lam, vec = np.linalg.eigh(Hp)
    u = vec[:, 0][:, None] * np.array([1.0, 0.5j, -0.25])[None, :]
    v, _ = plane_wave(dims, (1, 0, 3, 2), u, tb)
    coeff = inputs.chebyshev_sign_coefficients(30, 0.01)
    y = cplx(orc.cheb(real(v), inputs.unit_gauge_field(dims), dims, kappa, coeff, scale))
    want = np.polynomial.chebyshev.chebval(lam[0] / scale, coeff) * v
    assert relerr(y, want) < 1e-13


def test_chebyshev_coefficients_interpolate_the_smoothed_sign():
    deg, eps2 = 100, 0.01
    c = inputs.chebyshev_sign_coefficients(deg, eps2)
    N = deg + 1
    xj = np.cos(np.pi * (np.arange(N) + 0.5) / N)
    f = xj / np.sqrt(xj * xj + eps2)
    assert np.abs(np.polynomial.chebyshev.chebval(xj, c) - f).max() < 1e-13
    assert np.abs(c[0::2]).max() < 1e-13                                   # odd function


# ----------------------------------------------------------------------------- P11
def test_p11_mixed_cg_matches_pure_cg():
    dims, kappa = (4, 4, 4, 8), 0.1355
    U = inputs.gauge_field(dims, 0.5, seed=13)
    _, A, Ainv = clover_fields(U, dims, kappa, 1.0)
    b = inputs.spinor_field(dims, 13)
    for mode in (2, 0):
        bb = b if mode == 2 else b * (orc.parity_mask_array(dims) == 0)[..., None, None, None]
        x, st = orc.cg(bb, U, dims, kappa, 1e-10, 5000, A=A, Ainv=Ainv, mode=mode)
        y, sm = orc.cg_mixed(bb, U, dims, kappa, 1e-10, 5000, A=A, Ainv=Ainv, mode=mode)
        assert st["converged"] and sm["converged"]
        assert sm["r_true"] <= 1e-10 and st["r_true"] < 1.1e-10
        assert abs(sm["iters"] - st["iters"]) <= max(6, 0.08 * st["iters"])
        assert sm["reliable_updates"] >= 3
        assert relerr(y, x) < 1e-8


def dense_wilson_from_roll_stencil(U, dims, kappa):
    """192 x 192 matrix of 1 - kappa H on 2^4, column by column from the np.roll stencil above
    (written from the north_star formula; it shares nothing with the oracle)."""
    V = int(np.prod(dims)); n = 12 * V
    shape = (dims[3], dims[2], dims[1], dims[0], 4, 3)
    D = np.zeros((n, n), dtype=complex)
    e = np.zeros(n, dtype=complex)
    Uc = cplx(U)
    for j in range(n):
        e[:] = 0; e[j] = 1
        v = e.reshape(shape)
        D[:, j] = (v - kappa * roll_hop(v, Uc, dims, -1)).ravel()
    return D


def dense_reliable_update_cg(D, b, tol, maxiter, delta, track_rmax=True):
    """Reading O7 on dense matrices in numpy: inner x, r, p, q and N_lo in
    complex64, y / r_hi / N_hi in complex128, reductions accumulated in fp64.  Returns the iteration
    index of every reliable update.  track_rmax=False drops "rmax = max |r| since the last update"
    (the mutation VERDICT round 1 found unpinned) to show that the chosen cases depend on it."""
    Dl = D.astype(np.complex64)
    n2 = lambda v: float(np.vdot(v.astype(np.complex128), v.astype(np.complex128)).real)
    y = np.zeros(len(b), np.complex128); x = np.zeros(len(b), np.complex64)
    r = b.astype(np.complex64); p = r.copy()
    bnorm = np.sqrt(n2(b)); rho = n2(r); rmax = np.sqrt(rho)
    updates, k = [], 0
    while k < maxiter:
        k += 1
        q = Dl.conj().T @ (Dl @ p)
        pq = float(np.vdot(p.astype(np.complex128), q.astype(np.complex128)).real)
        alpha = np.float32(rho / pq)
        x = x + alpha * p; r = r - alpha * q
        rho2 = n2(r); rnorm = np.sqrt(rho2)
        if track_rmax and rnorm > rmax:
            rmax = rnorm
        if rnorm < delta * rmax or rnorm <= tol * bnorm:
            y = y + x.astype(np.complex128)
            rh = b - D.conj().T @ (D @ y)
            x = np.zeros_like(x); r = rh.astype(np.complex64)
            rho2 = n2(rh); rmax = np.sqrt(rho2)
            updates.append(k)
            if rmax <= tol * bnorm:
                break
        p = r + np.float32(rho2 / rho) * p
        rho = rho2
    return updates, y


@pytest.mark.parametrize("kappa,seed,delta,ncmp", [(0.22, 1, 0.5, 10), (0.20, 2, 0.1, 10), (0.19, 0, 0.5, 6)])
def test_p11_reliable_update_schedule_matches_dense_numpy_run(kappa, seed, delta, ncmp):
    """Pins O7's update rule -- rmax = max |r| since the last update, update when |r| < delta rmax --
    by the iteration indices of the reliable updates, against an independently written dense-matrix
    run (PAPER.md:163 ref. [1]).  The cases are ill-conditioned 2^4 systems
    (kappa near critical) whose fp32 residual rises above its value at the last update, so that
    dropping the running maximum, or using another delta, moves the updates; fp32 rounding differs
    between the two implementations, so only the first ncmp updates are compared."""
    dims = (2, 2, 2, 2)
    U = inputs.gauge_field(dims, 0.5, seed)
    D = dense_wilson_from_roll_stencil(U, dims, kappa)
    b = inputs.spinor_field(dims, seed, 1)
    bc = cplx(b).ravel()
    want, y_dense = dense_reliable_update_cg(D, bc, 1e-10, 3000, delta)
    mutant, _ = dense_reliable_update_cg(D, bc, 1e-10, 3000, delta, track_rmax=False)
    assert want[:ncmp] != mutant[:ncmp]                       # the case has teeth
    y, st = orc.cg_mixed(b, U, dims, kappa, 1e-10, 3000, delta=delta)
    assert st["converged"] and st["r_true"] <= 1e-10
    assert st["update_at"][:ncmp] == want[:ncmp]
    assert st["reliable_updates"] == len(st["update_at"])
    assert relerr(cplx(y).ravel(), np.linalg.solve(D.conj().T @ D, bc)) < 1e-7
    # another delta gives another schedule (delta is not ignored)
    _, st2 = orc.cg_mixed(b, U, dims, kappa, 1e-10, 3000, delta=0.5 if delta < 0.3 else 0.1)
    assert st2["update_at"][:3] != st["update_at"][:3]


# ---- multi-shift CG ----------------------------------------------------
def test_multishift_cg_matches_dense_shifted_solves_on_2to4():
    """Brute force: (D^dag D + sigma_i) x_i = b by LU on the 192 x 192 dense matrix."""
    dims, kappa = (2, 2, 2, 2), 0.135
    U = inputs.gauge_field(dims, 0.5, 0)
    D = dense_matrix(lambda v: orc.apply_M(v, U, dims, kappa), dims)
    N = D.conj().T @ D
    b = inputs.spinor_field(dims, 0, 1)
    shifts = [0.0, 0.01, 0.1, 1.0, 10.0]
    xs, st = orc.cg_multishift(b, U, dims, kappa, shifts, 1e-12, 1000)
    assert st["converged"] and not st["breakdown"]
    bc = cplx(b).reshape(-1)
    for x, sg in zip(xs, shifts):
        want = np.linalg.solve(N + sg * np.eye(N.shape[0]), bc)
        assert relerr(cplx(x).reshape(-1), want) < 1e-10
    assert st["r_true"].max() < 2e-12


def test_multishift_cg_reduces_to_plain_cg_and_each_shift_to_its_own_cg():
    dims, kappa = (4, 4, 4, 8), 0.135
    U = inputs.gauge_field(dims, 0.5, 0)
    _, A, Ainv = clover_fields(U, dims, kappa, 1.0)
    b = inputs.spinor_field(dims, 0, 1)
    x_ref, st_ref = orc.cg(b, U, dims, kappa, 1e-10, 2000, A, Ainv)
    # one shift equal to zero: the same iteration, iterate for iterate
    xs, st = orc.cg_multishift(b, U, dims, kappa, [0.0], 1e-10, 2000, A, Ainv)
    assert st["iters"] == st_ref["iters"]
    assert relerr(xs[0], x_ref) < 1e-13
    # several shifts: the unshifted member is unchanged, every member meets its residual,
    # and the shifted residuals obey |b - (N + s) x_s| <= |b - N x_0| (|zeta| <= 1)
    shifts = [0.0, 0.05, 0.5, 5.0]
    xs, st = orc.cg_multishift(b, U, dims, kappa, shifts, 1e-10, 2000, A, Ainv)
    assert st["iters"] == st_ref["iters"]
    assert relerr(xs[0], x_ref) < 1e-12
    assert (st["r_true"] < 1.5e-10).all()
    assert (st["r_true"][1:] <= st["r_true"][0] * 1.01).all()
    # non-zero base shift: compare with a dense-free identity, (N + s0) x = b  <=>  residual check
    xs2, st2 = orc.cg_multishift(b, U, dims, kappa, [0.5, 5.0], 1e-10, 2000, A, Ainv)
    assert relerr(xs2[0], xs[2]) < 1e-9 and relerr(xs2[1], xs[3]) < 1e-9
    assert st2["iters"] < st["iters"]


def test_multishift_cg_freezes_converged_shifts_on_a_long_solve():
    """Reading M1: a shifted system is frozen once |zeta_s| |r| <= tol |b|.  kappa = 0.2 on a random
    eps = 0.5 field needs ~470 iterations; zeta of the shift-10 system falls below 1e-154 after ~200,
    where the unfrozen recurrence's zeta^n zeta^{n-1} underflows and turns x_s into NaN.
    Every x_s must stay finite, meet its own residual, and agree with a CG run on N + sigma_s alone."""
    dims, kappa = (4, 4, 4, 8), 0.2
    U = inputs.gauge_field(dims, 0.5, 0)
    b = inputs.spinor_field(dims, 0, 1)
    shifts = [0.0, 1.0, 10.0]
    xs, st = orc.cg_multishift(b, U, dims, kappa, shifts, 1e-10, 5000)
    assert st["converged"] and st["iters"] > 300
    assert all(np.isfinite(x).all() for x in xs)
    assert (st["r_true"] < 1.5e-10).all()
    for x, sg in zip(xs[1:], shifts[1:]):
        x1, st1 = orc.cg_multishift(b, U, dims, kappa, [sg], 1e-12, 5000)
        assert st1["converged"] and relerr(x, x1[0]) < 1e-9
