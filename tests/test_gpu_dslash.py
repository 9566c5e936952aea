"""GPU parity: layout kernels, the hopping term, the clover term and the full / even-odd
operators, CUDA path (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Tolerances: BASELINE.json north_star (1e-12 fp64, 2e-6 fp32)."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2001_05706_b200 import inputs

from gpu_util import TOL, blocks, ctx, pack, parity_mask, relerr, to_dev, unpack

pytestmark = pytest.mark.gpu

# spans several 128-thread blocks with a ragged tail (Vh = 1536+..), tiny, L=2 wrap, odd X/2
DIMS = [(4, 4, 4, 4), (2, 2, 2, 2), (6, 4, 2, 8), (10, 6, 4, 12), (2, 8, 6, 4)]


def fields(dims, eps, precision, seed=0):
    U = inputs.gauge_field(dims, eps, seed)
    psi = inputs.spinor_field(dims, seed, 0)
    if precision == 4:
        U, psi = inputs.round_to_f32(U), inputs.round_to_f32(psi)
    return U, psi


@pytest.mark.parametrize("precision", [4, 8])
@pytest.mark.parametrize("dims", DIMS)
def test_spinor_pack_unpack_roundtrip_is_bit_exact(dims, precision):
    c = ctx()
    psi = inputs.spinor_field(dims, 3, 0)
    d = to_dev(psi, precision)
    internal = c.spinor_pack(d, dims)
    back = c.spinor_unpack(internal, dims)
    assert torch.equal(back, d)
    # internal layout = even block then odd block, [chunk][cb], chunk = 128 bits (include/qcd.h)
    X, Y, Z, T = dims
    Vh = X * Y * Z * T // 2
    rc = 16 // precision
    host = internal.cpu().numpy().reshape(2, 24 // rc, Vh, rc)
    flat = d.cpu().numpy().reshape(-1, 24)
    for (x, y, z, t) in [(0, 0, 0, 0), (X - 1, Y - 1, Z - 1, T - 1), (1, 0, 1, 1), (X - 2, 1, 0, T - 1)]:
        s = x + X * (y + Y * (z + Z * t))
        p, cb = (x + y + z + t) & 1, s >> 1
        assert np.array_equal(host[p, :, cb, :].reshape(24), flat[s])


@pytest.mark.parametrize("precision,recon", [(8, 18), (8, 12), (4, 18), (4, 12)])
@pytest.mark.parametrize("dims", DIMS)
@pytest.mark.parametrize("dagger", [False, True])
def test_hop_matches_oracle(dims, precision, recon, dagger):
    c = ctx()
    U, psi = fields(dims, 0.5, precision)
    g = c.gauge_load(to_dev(U, precision), dims, precision, recon, -1)
    pin = pack(c, psi, dims, precision)
    out = torch.zeros_like(pin)
    for p in (0, 1):
        c.hop(blocks(out)[p], blocks(pin)[1 - p], g, p, dagger)
    got = unpack(c, out, dims)
    want = orc.hop(psi, U, dims, -1, dagger, 2)
    assert relerr(got, want) <= TOL[precision]
    # one parity alone equals the oracle restricted to that parity
    m = parity_mask(dims)
    for p in (0, 1):
        want_p = orc.hop(psi, U, dims, -1, dagger, p)
        assert relerr(got * (m == p), want_p) <= TOL[precision]


def test_hop_periodic_t_boundary_and_xpay():
    c = ctx()
    dims, precision = (4, 6, 2, 8), 8
    U, psi = fields(dims, 0.5, precision)
    z = inputs.spinor_field(dims, 0, 5)
    g = c.gauge_load(to_dev(U, precision), dims, precision, 12, +1)
    pin, pz = pack(c, psi, dims, precision), pack(c, z, dims, precision)
    out = torch.zeros_like(pin)
    a, b = 0.75, -0.137
    for p in (0, 1):
        c.hop_xpay(blocks(out)[p], blocks(pin)[1 - p], blocks(pz)[p], a, b, g, p, False)
    want = a * z + b * orc.hop(psi, U, dims, +1, False, 2)
    assert relerr(unpack(c, out, dims), want) <= TOL[precision]


def test_config0_wilson_4to4_fp64_full_lattice():
    """BASELINE.json configs[0]: 4^4, fp64, eps 0.3, kappa 0.125, antiperiodic t, seed 0."""
    c = ctx()
    dims, kappa = (4, 4, 4, 4), 0.125
    U = inputs.gauge_field(dims, 0.3, 0)
    psi = inputs.spinor_field(dims, 0, 0)
    for recon in (18, 12):
        g = c.gauge_load(to_dev(U, 8), dims, 8, recon, -1)
        pin = pack(c, psi, dims, 8)
        out = torch.empty_like(pin)
        c.dslash(out, pin, g, None, kappa, 0.0, 2)
        want = orc.apply_M(psi, U, dims, kappa)
        assert relerr(unpack(c, out, dims), want) <= 1e-12


def oracle_clover(U, dims, kappa, csw):
    F = orc.field_strength(U, dims)
    A = orc.clover_matrix(F, dims, kappa * csw)
    return A, orc.invert_12(A)


@pytest.mark.parametrize("precision", [8, 4])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (2, 2, 2, 2), (6, 4, 2, 8)])
def test_clover_build_matches_oracle(dims, precision):
    c = ctx()
    kappa, csw = 0.135, 1.0
    U = inputs.gauge_field(dims, 0.5, 0)
    A, Ainv = oracle_clover(U, dims, kappa, csw)
    for recon in (18, 12):
        g = c.gauge_load(to_dev(U, 8), dims, 8, recon, -1)
        cl = c.clover_build(g, kappa, csw, precision)
        gotA = c.clover_unpack(cl, 0).cpu().numpy()
        gotI = c.clover_unpack(cl, 1).cpu().numpy()
        assert relerr(gotA, A) <= TOL[precision]
        assert relerr(gotI, Ainv) <= TOL[precision]


@pytest.mark.parametrize("precision,recon", [(8, 18), (4, 12)])
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8), (10, 6, 4, 12)])
@pytest.mark.parametrize("clover", [False, True])
@pytest.mark.parametrize("dagger", [False, True])
def test_full_and_even_odd_operator_match_oracle(dims, precision, recon, clover, dagger):
    c = ctx()
    kappa, csw = 0.135, 1.0
    U, psi = fields(dims, 0.5, precision)
    g = c.gauge_load(to_dev(U, precision), dims, precision, recon, -1)
    A = Ainv = cl = None
    if clover:
        # the clover field is built in fp64 from the links the operator uses, stored in `precision`
        cl = c.clover_build(g, kappa, csw, precision)
        A, Ainv = oracle_clover(U, dims, kappa, csw)
        if precision == 4:
            A, Ainv = inputs.round_to_f32(A), inputs.round_to_f32(Ainv)
    pin = pack(c, psi, dims, precision)
    flags = 1 if dagger else 0
    # full lattice
    out = torch.empty_like(pin)
    c.dslash_ex(out, pin, g, cl, kappa, csw if clover else 0.0, 2, flags)
    want = orc.apply_M(psi, U, dims, kappa, A, Ainv, -1, 2, dagger)
    assert relerr(unpack(c, out, dims), want) <= TOL[precision]
    # even-odd Schur operator on each parity
    m = parity_mask(dims)
    tmp = torch.empty_like(blocks(pin)[0])
    for p in (0, 1):
        full = torch.zeros_like(pin)
        c.dslash_ex(blocks(full)[p], blocks(pin)[p], g, cl, kappa, csw if clover else 0.0, p, flags, tmp)
        want = orc.apply_M(psi * (m == p), U, dims, kappa, A, Ainv, -1, p, dagger)
        assert relerr(unpack(c, full, dims), want) <= TOL[precision]


def test_argument_errors_are_reported():
    from paper_2001_05706_b200 import qcd
    c = ctx()
    dims = (4, 4, 4, 4)
    U, psi = fields(dims, 0.5, 8)
    g = c.gauge_load(to_dev(U, 8), dims, 8, 18, -1)
    pin = pack(c, psi, dims, 8)
    with pytest.raises(qcd.QcdError) as e:
        c.hop(blocks(pin)[0], blocks(pin)[0], g, 0)          # aliased
    assert e.value.code == qcd.EINVAL
    with pytest.raises(qcd.QcdError):
        c.hop(blocks(pin)[0][1:], blocks(pin)[1], g, 0)      # misaligned
    with pytest.raises(qcd.QcdError):
        c.gauge_load(to_dev(U, 8), (3, 4, 4, 4), 8, 18, -1)  # odd extent
    cl = c.clover_build(g, 0.135, 1.0, 8)
    out = torch.empty_like(pin)
    with pytest.raises(qcd.QcdError):
        c.dslash(out, pin, g, cl, 0.136, 1.0, 2)             # kappa differs from the clover's (S10)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (6, 4, 2, 8)])
def test_convert_is_layout_aware(dims):
    """fp32 <-> fp64 conversion of internal fields keeps (site, spin, colour) in place."""
    c = ctx()
    psi = inputs.spinor_field(dims, 1, 0)
    p64 = pack(c, psi, dims, 8)
    p32 = c.convert(p64, 4, dims, 2)
    assert torch.equal(c.spinor_unpack(p32, dims), to_dev(psi, 8).float())
    back = c.convert(p32, 8, dims, 2)
    assert torch.equal(c.spinor_unpack(back, dims), to_dev(psi, 8).float().double())
    h = p64.numel() // 2
    one = c.convert(p64[h:], 4, dims, 1)
    assert torch.equal(one, p32[h:])


def test_dslash_host_batch_matches_single_calls():
    """qcd_dslash_host_batch (pipelined copies on the ctx's own copy streams) gives, vector by vector,
    the bits qcd_dslash_host gives; covers nvec = 0, 1 and an odd count (both double buffers reused)."""
    from paper_2001_05706_b200 import qcd
    c = ctx()
    dims, kappa, csw = (8, 6, 4, 10), 0.135, 1.0
    U = inputs.gauge_field(dims, 0.5, 0)
    g = c.gauge_load(to_dev(U, 4), dims, 4, 12, -1)
    g64 = c.gauge_load(to_dev(U, 8), dims, 8, 18, -1)
    cl = c.clover_build(g64, kappa, csw, 4)
    V = int(np.prod(dims))
    for parity, n in ((0, V // 2 * 24), (2, V * 24)):
        c.set_workspace(None)
        c.ensure_workspace(5 * n * 4)
        for nvec in (0, 1, 5):
            hin = torch.randn(max(nvec, 1) * n, dtype=torch.float32, generator=torch.Generator().manual_seed(nvec)).pin_memory()
            hout = torch.zeros(max(nvec, 1) * n, dtype=torch.float32).pin_memory()
            c.dslash_host_batch(hout, hin, nvec, g, cl, kappa, csw, parity, 0, out_stride=n * 4, in_stride=n * 4)
            one = torch.zeros(n, dtype=torch.float32).pin_memory()
            for i in range(nvec):
                c.dslash_host(one, hin[i * n:(i + 1) * n], g, cl, kappa, csw, parity, 0)
                assert torch.equal(one, hout[i * n:(i + 1) * n])
            if nvec == 0:
                assert float(hout.abs().max()) == 0.0
    with pytest.raises(qcd.QcdError):
        c.dslash_host_batch(hout, hin, 2, g, cl, kappa, csw, 2, 0, out_stride=16, in_stride=n * 4)
    c.set_workspace(None)


@pytest.mark.parametrize("precision", [4, 8])
@pytest.mark.parametrize("dims,nvec", [((4, 4, 4, 4), 1), ((6, 4, 2, 8), 3), ((10, 6, 4, 12), 2)])
def test_wilson_multi_matches_oracle(dims, nvec, precision):
    """qcd_wilson_multi (links fetched once per block for all right-hand sides):
    every vector against the oracle's D_W and gamma5 D_W."""
    c = ctx()
    kappa = 0.137
    U, _ = fields(dims, 0.5, precision)
    g = c.gauge_load(to_dev(U, precision), dims, precision, 12 if precision == 4 else 18, -1)
    vs = [inputs.spinor_field(dims, 0, 40 + i) for i in range(nvec)]
    if precision == 4:
        vs = [inputs.round_to_f32(v) for v in vs]
    batch = torch.cat([pack(c, v, dims, precision) for v in vs])
    n = batch.numel() // nvec
    for gamma5 in (False, True):
        out = torch.empty_like(batch)
        c.wilson_multi(out, batch, nvec, g, kappa, gamma5)
        for i, v in enumerate(vs):
            want = orc.apply_HW(v, U, dims, kappa) if gamma5 else orc.apply_M(v, U, dims, kappa)
            assert relerr(unpack(c, out[i * n:(i + 1) * n].contiguous(), dims), want) <= TOL[precision]
    from paper_2001_05706_b200 import qcd
    with pytest.raises(qcd.QcdError):
        c.wilson_multi(batch, batch, nvec, g, kappa)          # aliased


def test_clover_build_reports_a_block_it_cannot_invert():
    """A non-finite pivot of the L D L^dag factorisation (here from a NaN link) is QCD_EBREAKDOWN, not a silent
    NaN field; an ordinary field on the same lattice still builds afterwards."""
    from paper_2001_05706_b200 import qcd
    c = ctx()
    dims = (4, 4, 4, 4)
    U = inputs.gauge_field(dims, 0.5, 0)
    bad = U.copy()
    bad[0, 1, 2, 3, 0, 0, 0, 0] = np.nan
    g = c.gauge_load(to_dev(bad, 8), dims, 8, 18, -1)
    with pytest.raises(qcd.QcdError) as e:
        c.clover_build(g, 0.135, 1.0, 8)
    assert e.value.code == qcd.EBREAKDOWN
    g = c.gauge_load(to_dev(U, 8), dims, 8, 18, -1)
    cl = c.clover_build(g, 0.135, 1.0, 8)
    A, Ainv = oracle_clover(U, dims, 0.135, 1.0)
    assert relerr(c.clover_unpack(cl, 1).cpu().numpy(), Ainv) <= 1e-12


def test_even_odd_operator_can_be_captured_in_a_cuda_graph():
    """SURVEY 8(d) caveat (i): at small sizes the launches are what costs; the operator (launched with programmatic
    stream serialisation) captures into a CUDA graph on the ctx's stream and the replay gives the eager bits."""
    from paper_2001_05706_b200 import qcd
    dims, kappa, csw = (8, 8, 8, 16), 0.135, 1.0
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        c = qcd.Context(0, stream=s)
        U = inputs.round_to_f32(inputs.gauge_field(dims, 0.5, 0))
        g = c.gauge_load(to_dev(U, 4), dims, 4, 12, -1)
        cl = c.clover_build(g, kappa, csw, 4)
        pin = c.spinor_pack(to_dev(inputs.round_to_f32(inputs.spinor_field(dims, 0, 0)), 4), dims)
        h = pin.numel() // 2
        src, mid, dst, tmp = pin[:h].clone(), torch.empty_like(pin[:h]), torch.empty_like(pin[:h]), torch.empty_like(pin[:h])
        c.dslash_ex(mid, src, g, cl, kappa, csw, 0, 0, tmp)
        c.dslash_ex(dst, mid, g, cl, kappa, csw, 0, qcd.DAGGER, tmp)      # dst = Mhat^dag Mhat src, eagerly
    s.synchronize()
    want = dst.clone()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=s):
        c.dslash_ex(mid, src, g, cl, kappa, csw, 0, 0, tmp)
        c.dslash_ex(dst, mid, g, cl, kappa, csw, 0, qcd.DAGGER, tmp)
    dst.zero_()
    mid.zero_()
    torch.cuda.synchronize()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(dst, want)
    src.mul_(2.0)
    torch.cuda.synchronize()
    graph.replay()
    torch.cuda.synchronize()
    assert torch.equal(dst, 2.0 * want)
    del graph
    c.close()
