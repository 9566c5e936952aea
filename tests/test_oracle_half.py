"""Pins of the 16-bit storage format of the low-precision operator (reading H1
in DESIGN.md): hand-computed codes, the error bound of the format, structure preserved by the
link / clover storage, the size of the operator's storage error, and convergence of the
reliable-update CG whose inner operator streams 16-bit fields."""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2001_05706_b200 import inputs


def cplx(a):
    return a[..., 0] + 1j * a[..., 1]


def relerr(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return float(np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel()))


def test_spinor_codes_by_hand():
    # n = 2: scale = 32767/2; 2 -> 32767, -1 -> -16383.5 -> -16384 (ties to even), 0.5 -> 8191.75 -> 8192,
    # 1e-5 -> 0.1638 -> 0, -2 -> -32767
    v = np.zeros((2, 24), dtype=np.float32)
    v[0, :5] = [2.0, -1.0, 0.5, 1e-5, -2.0]
    codes, norms = orc.q16_codes(v)
    assert list(codes[0, :5]) == [32767, -16384, 8192, 0, -32767] and norms[0] == 2.0
    assert not codes[1].any() and norms[1] == 0.0          # an all-zero site stays zero
    back = orc.q16_spinor(v)
    assert back[0, 0] == np.float32(32767) * (np.float32(2.0) / np.float32(32767.0))
    assert not back[1].any()


def test_spinor_storage_error_bound_and_sign_symmetry():
    rng = np.random.default_rng(1)
    v = (rng.standard_normal((4096, 24)) * np.exp(rng.uniform(-8, 8, (4096, 1)))).astype(np.float32)
    back = orc.q16_spinor(v)
    n = np.abs(v).max(axis=1, keepdims=True)
    assert (np.abs(back - v) <= n / 65534.0 + 3e-7 * n).all()        # half a code step + fp32 rounding
    assert np.array_equal(orc.q16_spinor(-v), -back)
    codes, norms = orc.q16_codes(v)
    assert np.array_equal(norms, n[:, 0]) and np.abs(codes).max() == 32767


def test_link_storage_keeps_su3_to_format_accuracy():
    dims = (4, 4, 4, 4)
    U = inputs.gauge_field(dims, 0.5, 0)
    Uq = orc.q16_links(U)
    u, uq = cplx(U).reshape(-1, 3, 3), cplx(Uq.astype(np.float64)).reshape(-1, 3, 3)
    assert np.abs(uq[:, :2] - u[:, :2]).max() <= 0.5 / 32767 * np.sqrt(2) * 1.001      # rows 0,1: half a step per real
    # row 2 is rebuilt from the stored rows, not stored: exactly conj(r0 x r1) of the stored values
    assert np.abs(uq[:, 2] - np.conj(np.cross(uq[:, 0], uq[:, 1]))).max() < 2e-7
    eye = np.eye(3)
    assert np.abs(uq @ np.conj(np.swapaxes(uq, 1, 2)) - eye).max() < 2e-4
    assert np.abs(np.linalg.det(uq) - 1).max() < 2e-4


def test_clover_storage_is_hermitian_block_diagonal_and_close():
    dims, kappa = (4, 4, 2, 2), 0.135
    U = inputs.gauge_field(dims, 0.5, 0)
    A = orc.clover_matrix(orc.field_strength(U, dims), dims, kappa)
    Aq = cplx(orc.q16_clover(A).astype(np.float64)).reshape(-1, 12, 12)
    a = cplx(A).reshape(-1, 12, 12)
    assert np.array_equal(Aq, np.conj(np.swapaxes(Aq, 1, 2)))
    assert not Aq[:, :6, 6:].any() and not Aq[:, 6:, :6].any()
    n = np.maximum(np.abs(a.real), np.abs(a.imag)).max(axis=(1, 2), keepdims=True)
    assert (np.abs(Aq - a) <= n / 65534.0 * np.sqrt(2) * 1.001 + 1e-7).all()


@pytest.mark.parametrize("mode", [2, 0])
def test_operator_storage_error_is_small_but_present(mode):
    dims, kappa, csw = (4, 4, 4, 8), 0.1355, 1.0
    U = inputs.gauge_field(dims, 0.5, 0)
    A = orc.clover_matrix(orc.field_strength(U, dims), dims, kappa * csw)
    Ainv = orc.invert_12(A)
    p = inputs.spinor_field(dims, 0, 1)
    if mode == 0:
        p = p * (orc.parity_mask_array(dims) == 0)[..., None, None, None]
    want = orc.apply_M(orc.apply_M(p, U, dims, kappa, A, Ainv, -1, mode), U, dims, kappa, A, Ainv, -1, mode, True)
    got = orc.apply_N_q16(p, orc.q16_links(U), dims, kappa, orc.q16_clover(A), orc.q16_clover(Ainv), -1, mode)
    e = relerr(got, want)
    assert 2e-6 < e < 3e-4


@pytest.mark.parametrize("mode", [2, 0])
def test_half_mixed_cg_converges_like_the_fp64_cg(mode):
    dims, kappa, csw, tol = (4, 4, 4, 8), 0.1355, 1.0, 1e-10
    U = inputs.gauge_field(dims, 0.5, 0)
    A = orc.clover_matrix(orc.field_strength(U, dims), dims, kappa * csw)
    Ainv = orc.invert_12(A)
    b = inputs.spinor_field(dims, 0, 1)
    if mode == 0:
        b = b * (orc.parity_mask_array(dims) == 0)[..., None, None, None]
    x64, st64 = orc.cg(b, U, dims, kappa, tol, 5000, A, Ainv, -1, mode)
    y, st = orc.cg_mixed(b, U, dims, kappa, tol, 5000, A, Ainv, -1, mode, 0.1, half=True)
    assert st["converged"] and st["r_true"] <= 1.01 * tol          # fp64 true residual, recomputed
    assert relerr(y, x64) < 1e-8
    assert st["iters"] <= 1.5 * st64["iters"] + 5
    assert st["reliable_updates"] >= 8
