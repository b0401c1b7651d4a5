"""moto_gram_static (csrc/gram_static.cu): the Gram product with its reduction scratch in a file-scope __device__ array -- no
context, no workspace, no cudaMalloc -- against the existing path moto_gram on the same inputs, two calls in a row (the second
call finds the first call's partial sums and ticket in the shared array).  Collected last (file name), so a failure here hides
no other test under `pytest -x`; passes alone in a fresh process and after the other tests.  Tolerance: test_gram_parity's."""
import numpy as np
import pytest

from paper_2509_26269_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def close(G, ref):
    return np.max(np.abs(G - ref)) <= 1e-11 * np.max(np.abs(ref)) + 1e-10


def test_gram_static_matches_moto_gram_two_calls(moto):
    import torch
    w = wl.SpinWorkload("rand50x41", 50, 41, 1, 1, 1.0, 0.3, 0.05, (0.01, -0.02, 0.03), 1.0, 2, 9, wl.random_spins(50, 41, 9))
    ctx = moto.spin_context(w, kmax=8)
    G = torch.full((6, 12), float("nan"), dtype=torch.float64, device="cuda")     # caller-owned output, reused
    # call 1: the full 6 x 12 pencil on a lattice with a ragged last chunk (3 N = 6150 = 96 chunks of 64 + 6)
    S1, T1 = dev(wl.random_block(w.N, 6, seed=1)), dev(wl.random_block(w.N, 12, seed=2))
    ref1 = ctx.gram(S1, T1).cpu().numpy()
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    moto.gram_static(S1, T1, G)
    got1 = G.cpu().numpy().copy()
    # call 2, straight after: other data, smaller pencil (stale partials of call 1 sit beside the ones it uses)
    S2, T2 = dev(wl.random_block(w.N, 6, seed=3))[:3].contiguous(), dev(wl.random_block(w.N, 12, seed=4))[:5].contiguous()
    ref2 = ctx.gram(S2, T2).cpu().numpy()
    torch.cuda.synchronize()
    G2 = G.view(-1)[:15].view(3, 5)
    moto.gram_static(S2, T2, G2)
    got2 = G2.cpu().numpy().copy()
    # call 3 = call 1 again: bit-identical (fixed summation order, nothing left over from call 2)
    moto.gram_static(S1, T1, G)
    got3 = G.cpu().numpy()
    assert torch.cuda.mem_get_info()[0] >= free0, "device memory shrank across moto_gram_static calls"
    host1 = S1.cpu().numpy().reshape(6, -1) @ T1.cpu().numpy().reshape(12, -1).T
    assert close(got1, ref1) and close(got1, host1)
    assert close(got2, ref2)
    assert np.array_equal(got1, got3)


def test_gram_static_large_and_tiny(moto):
    import torch
    # more chunks than CTAs (every CTA strides), and a single partial chunk (one CTA, ticket 0 = last)
    for n3, ns, nt, seed in ((3 * 400 * 400, 2, 4, 5), (7, 1, 1, 6)):
        rng = np.random.default_rng(seed)
        S, T = rng.standard_normal((ns, n3)), rng.standard_normal((nt, n3))
        G = torch.empty((ns, nt), dtype=torch.float64, device="cuda")
        moto.gram_static(dev(S), dev(T), G)
        assert close(G.cpu().numpy(), S @ T.T)


def test_gram_static_rejects_sizes_beyond_the_scratch(moto):
    import torch
    S, T = torch.zeros((7, 30), dtype=torch.float64, device="cuda"), torch.zeros((13, 30), dtype=torch.float64, device="cuda")
    G = torch.zeros((7, 13), dtype=torch.float64, device="cuda")
    with pytest.raises(moto.MotoError, match="beyond the static scratch"):
        moto.gram_static(S, T[:12].contiguous(), G[:, :12].contiguous())
    with pytest.raises(moto.MotoError, match="beyond the static scratch"):
        moto.gram_static(S[:6].contiguous(), T, G[:6].contiguous())
    torch.cuda.synchronize()
