"""leb_jerr_static (include/leb.h): the propagated-error penalty (35) PAPER.md:L360 for callers that cannot allocate.
Its per-(b, j) partial sums live in a static device array of the library instead of a cudaMalloc'ed buffer.  Checked
here against the existing path leb_jerr on two calls in a row (the second smaller, so stale contents of the shared
array would show), at the tolerance of the tube tests; capacity and host-IO rejections; no change of the device's free
memory across a call.  Collected last on purpose (the file name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from parity_util import BOUND_ATOL, BOUND_RTOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def leb():
    from paper_2607_01203_b200 import build, leb as L
    build.build()
    return L


def _case(seed, B, T, n, m):
    g = torch.Generator(device="cuda")
    g.manual_seed(seed)
    nb = T * (T + 1) // 2
    Phi = torch.randn((B, nb, n + m, n), device="cuda", generator=g) / n ** 0.5
    for j in range(T):
        Phi[:, (j + 1) * j // 2 + j, :n] = torch.eye(n, device="cuda")          # Phi^x_{j+1,j} = I (34c)
    R = torch.rand((B, T, n), device="cuda", generator=g) * 0.1 + 1e-3
    E = torch.rand((n,), device="cuda", generator=g) * 0.05
    return Phi, R, E


def _close(a, b):
    return bool(((a - b).abs() <= BOUND_RTOL * b.abs() + BOUND_ATOL).all())


def test_jerr_static_matches_jerr_two_calls_in_a_row(leb):
    ctx = leb.Context(0)
    cases = [(_case(1, 3, 9, 168, 56), 56), (_case(2, 2, 4, 33, 0), 0)]        # vectorised and scalar loads; second is smaller
    outs = [(torch.full((c[1].shape[0],), -7.0, device="cuda"), torch.full(tuple(c[1].shape), -7.0, device="cuda")) for c, _ in cases]
    ref = [ctx.leb_jerr(Phi, R, m, E) for (Phi, R, E), m in cases]              # the existing path (allocates its scratch)
    torch.cuda.synchronize()
    # warm-up of the entry point itself (module / kernel loading), then the two calls in a row with no allocation between
    ctx.leb_jerr_static(cases[0][0][0], cases[0][0][1], cases[0][1], outs[0][0], outs[0][1], E_diag=cases[0][0][2])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for ((Phi, R, E), m), (J, g) in zip(cases, outs):
        J.fill_(-7.0); g.fill_(-7.0)
        ctx.leb_jerr_static(Phi, R, m, J, g, E_diag=E)
    torch.cuda.synchronize()
    assert free0 - torch.cuda.mem_get_info()[0] < (2 << 20)                    # the device's free memory did not drop (2 MiB: the driver's granularity)
    for (J, g), (Jr, gr) in zip(outs, ref):
        assert _close(J, Jr) and _close(g, gr)
        assert torch.equal(J, Jr) and torch.equal(g, gr)                        # same kernels, same order: bit for bit
    # without the gradient, without E
    (Phi, R, E), m = cases[1]
    J = torch.empty((R.shape[0],), device="cuda")
    ctx.leb_jerr_static(Phi, R, m, J)
    Jr, _ = ctx.leb_jerr(Phi, R, m, None, with_grad=False)
    assert _close(J, Jr)
    ctx.close()


def test_jerr_static_rejects_what_it_cannot_hold(leb):
    ctx = leb.Context(0)
    B, T, n = 257, 256, 4                                                      # B * T = 65 792 > 65 536
    assert B * T > leb.JERR_STATIC_MAX
    Phi = torch.zeros((1,), device="cuda")                                     # never read: the call is refused before any launch
    R = torch.zeros((B, T, n), device="cuda")
    J = torch.zeros((B,), device="cuda")
    with pytest.raises(leb.LebError) as e:
        ctx.leb_jerr_static(Phi, R, 0, J)
    assert e.value.status == leb.LEB_ERR_CAPACITY
    R2 = torch.zeros((2, 3, n), device="cuda")
    with pytest.raises(leb.LebError) as e:
        ctx.leb_jerr_static(Phi, R2, 0, J, flags=leb.FLAG_HOST_IO)
    assert e.value.status == leb.LEB_ERR_ARG
    ctx.close()
