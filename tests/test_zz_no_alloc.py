"""qcd_norm2_noalloc (include/qcd.h): the reduction whose scratch is a static device array, against the
existing qcd_norm2 path, on calls in a row that share that array.  Collected last on purpose (file name)."""
import numpy as np
import pytest
import torch

from paper_2001_05706_b200 import qcd

from gpu_util import ctx

pytestmark = pytest.mark.gpu

RTOL = 1e-13   # the tolerance tests/test_gpu_solvers.py::test_blas_matches_numpy_fp64 holds qcd_norm2 to


def field(n, precision, seed):
    rng = np.random.default_rng(seed)
    return torch.from_numpy(rng.standard_normal(n).astype({4: np.float32, 8: np.float64}[precision])).cuda()


@pytest.mark.parametrize("precision", [4, 8])
def test_norm2_noalloc_matches_qcd_norm2_on_calls_in_a_row(precision):
    c = ctx()
    qcd.noalloc_setup(0)
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda")
    # a large field first (1465 blocks' partials left behind), then a short ragged one, then a mid-sized one,
    # then the first again: every call finds the previous call's partials and a used ticket in the array
    sizes = [24 * 250000, 24 * 1000 + 4, 24 * 8 * 8 * 8 * 16, 24 * 250000]
    xs = [field(n, precision, 100 + i) for i, n in enumerate(sizes[:3])]
    xs.append(xs[0])
    want = [c.norm2(x) for x in xs]
    got = []
    for x in xs:
        qcd.norm2_noalloc(x, out[:1])
        qcd.norm2_noalloc(x, out[1:])          # twice in a row on the same stream
        torch.cuda.synchronize()
        a, b = out.tolist()
        assert a == b                          # deterministic, whatever the array held before
        got.append(a)
    for g, w, x in zip(got, want, xs):
        assert abs(g - w) <= RTOL * w
        x64 = x.double().cpu().numpy()
        assert abs(g - np.dot(x64, x64)) <= RTOL * np.dot(x64, x64)
    assert got[0] == got[3]


def test_norm2_noalloc_allocates_nothing_and_rejects_what_the_scratch_cannot_cover():
    qcd.noalloc_setup(0)
    x = field(24 * 100000, 4, 7)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    qcd.norm2_noalloc(x, out)                  # first launch: the kernel's code is loaded now
    torch.cuda.synchronize()
    unchanged = False
    for _ in range(3):                         # free device memory is global to the GPU: allow for an unrelated change
        free0, _ = torch.cuda.mem_get_info()
        for _ in range(3):
            qcd.norm2_noalloc(x, out)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        unchanged = unchanged or free1 == free0
    assert unchanged
    limit = qcd.noalloc_max_bytes()
    assert limit == 1 << 30
    before = out.clone()
    with pytest.raises(qcd.QcdError) as e:     # the size is checked before anything is enqueued or read
        qcd.norm2_noalloc(x, out, nreal=limit // 4 + 4)
    assert e.value.code == qcd.EINVAL and "exceed" in str(e.value)
    with pytest.raises(qcd.QcdError):
        qcd.norm2_noalloc(x, out, nreal=6)     # not a whole number of 128-bit words
    torch.cuda.synchronize()
    assert torch.equal(out, before)
    qcd.norm2_noalloc(x, out, nreal=limit // 4 // 1024)   # a size at which the limit check passes still works
    torch.cuda.synchronize()
    part = x[: limit // 4 // 1024].double().cpu().numpy()
    assert abs(out.item() - np.dot(part, part)) <= RTOL * np.dot(part, part)


def test_norm2_noalloc_can_be_captured_in_a_cuda_graph_and_replayed():
    """What the entry point is for: it runs under stream capture (nothing in it allocates or synchronises) and the
    replayed graph recomputes from the current contents of x."""
    qcd.noalloc_setup(0)                       # set-up belongs outside the capture
    x = field(24 * 100000, 4, 11)
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        qcd.norm2_noalloc(x, out)              # uncaptured call on the same stream: loads the kernel, gives the value
    s.synchronize()
    want = out.item()
    x64 = x.double().cpu().numpy()
    assert abs(want - np.dot(x64, x64)) <= RTOL * want
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        qcd.norm2_noalloc(x, out)
    out.zero_()
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    assert out.item() == want
    x.mul_(2.0)                                # exact in binary: the sum of squares scales by exactly 4
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    assert out.item() == 4.0 * want
