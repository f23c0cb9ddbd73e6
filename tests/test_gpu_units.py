"""-m gpu: single kernels of the path against the oracle / plain references, through the C ABI."""
import os

import numpy as np
import pytest
import torch

import paper_2606_28166_b200 as T
from oracle import rng as orng

pytestmark = pytest.mark.gpu
GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def test_philox_known_answers_on_device():
    for line in open(GOLDEN):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        r = line.split()
        ins = [int(x, 16) for x in r[:6]]
        out = T.tandem_test_philox(ins[:4], ins[4:])
        for got, exp in zip(out, r[6:]):
            if "?" not in exp:
                assert got == int(exp, 16)


@pytest.mark.parametrize("seed", [0, 7, (1 << 40) + 12345])
def test_uniforms_bit_identical_to_oracle(seed):
    """Pin 14: the two independently written generators agree bit for bit on > 10^6 values."""
    n = 151936
    out = torch.empty(n, dtype=torch.float32, device="cuda")
    total = 0
    for (b, t) in [(0, 1), (3, 17), (127, 4096), (511, 8192), (1000003, 2), (5, 5), (6, 6), (9, 999)]:
        T.tandem_test_uniforms(seed, b, t, 0, n, out)
        ref = orng.uniforms_sample(seed, b, t, n)
        assert np.array_equal(out.cpu().numpy().view(np.uint32), ref.view(np.uint32))
        total += n
    assert total > 10 ** 6
    sw = torch.empty(4097, dtype=torch.float32, device="cuda")
    for b in (0, 1, 77):
        T.tandem_test_uniforms(seed, b, 0, 1, 4097, sw)
        ref = np.array([orng.uniforms_switch(seed, b, t) for t in range(0, 4097, 64)], dtype=np.float32)
        assert np.array_equal(sw.cpu().numpy()[::64].view(np.uint32), ref.view(np.uint32))


@pytest.mark.parametrize("rows,N,K", [(1, 32, 32), (7, 96, 128), (33, 512, 128), (129, 1152, 896), (64, 40, 72)])
def test_simt_gemm_fp32(rows, N, K):
    g = torch.Generator().manual_seed(rows * 1000 + N)
    A = torch.randn(rows, K, generator=g).cuda()
    W = (torch.randn(N, K, generator=g) * 0.05).cuda()
    out = torch.zeros(rows, N, device="cuda")
    T.tandem_test_gemm(T.F32, T.GEMM_SIMT, A, W, out)
    ref = (A.double() @ W.double().T)
    assert torch.max(torch.abs(out.double() - ref)).item() <= 2e-6 * max(1.0, ref.abs().max().item()) * (K ** 0.5)


@pytest.mark.parametrize("rows,N,K", [(5, 64, 64), (130, 1152, 896)])
def test_simt_gemm_bf16(rows, N, K):
    g = torch.Generator().manual_seed(rows + N)
    A = torch.randn(rows, K, generator=g).to(torch.bfloat16).cuda()
    W = (torch.randn(N, K, generator=g) * 0.05).to(torch.bfloat16).cuda()
    out = torch.zeros(rows, N, device="cuda")
    T.tandem_test_gemm(T.BF16, T.GEMM_SIMT, A, W, out)
    ref = (A.double() @ W.double().T)
    assert torch.max(torch.abs(out.double() - ref)).item() <= 2e-6 * max(1.0, ref.abs().max().item()) * (K ** 0.5)


@pytest.mark.parametrize("rows,N,K", [(1, 128, 64), (7, 256, 128), (32, 128, 256), (33, 384, 192), (64, 512, 256), (128, 6144, 2560),
                                      (129, 2560, 4096), (300, 1152, 896), (256, 2560, 9728), (257, 1024, 512), (61, 4096, 2560),
                                      (5, 200, 72), (1000, 640, 1024)])
def test_tcgen05_gemm_bf16(rows, N, K):
    """tcgen05/TMEM/TMA GEMM (swap-AB, split-K) against a float64 matmul of the same bf16 values: the seven projection
    shapes of the configs plus ragged rows (1, 33, 257, 1000), N not a multiple of the 128-row tile and K not a multiple of 64.
    Also as CTA pairs (cta_group::2, impl 4): same accumulation order per output, so bit-identical to the single-CTA kernel."""
    g = torch.Generator().manual_seed(rows * 7919 + N + K)
    A = torch.randn(rows, K, generator=g).to(torch.bfloat16).cuda()
    W = (torch.randn(N, K, generator=g) * 0.05).to(torch.bfloat16).cuda()
    out = torch.full((rows, N), float("nan"), device="cuda")
    T.tandem_test_gemm(T.BF16, T.GEMM_TCGEN05, A, W, out)
    ref = (A.double() @ W.double().T)
    err = torch.max(torch.abs(out.double() - ref)).item()
    assert np.isfinite(err)
    assert err <= 2e-6 * max(1.0, ref.abs().max().item()) * (K ** 0.5), (err, ref.abs().max().item())
    pair = torch.full((rows, N), float("nan"), device="cuda")
    T.tandem_test_gemm(T.BF16, 4, A, W, pair)
    assert torch.equal(pair, out)


@pytest.mark.parametrize("rows,I,K", [(1, 64, 64), (37, 192, 128), (140, 9728, 2560), (300, 512, 256), (64, 4864, 896)])
def test_tcgen05_gemm_swiglu_epilogue(rows, I, K):
    """Gate/up projection with SwiGLU fused into the tcgen05 epilogue (rows of W interleaved gate/up) against float64."""
    g = torch.Generator().manual_seed(rows * 31 + I + K)
    A = torch.randn(rows, K, generator=g).to(torch.bfloat16).cuda()
    Wg = (torch.randn(I, K, generator=g) * 0.05).to(torch.bfloat16)
    Wu = (torch.randn(I, K, generator=g) * 0.05).to(torch.bfloat16)
    W = torch.stack([Wg, Wu], dim=1).reshape(2 * I, K).contiguous().cuda()
    out = torch.zeros(rows, I, dtype=torch.bfloat16, device="cuda")
    T.tandem_test_gemm(T.BF16, 3, A, W, out)
    gate = A.double() @ Wg.cuda().double().T
    up = A.double() @ Wu.cuda().double().T
    ref = gate / (1 + torch.exp(-gate)) * up
    err = torch.max(torch.abs(out.double() - ref)).item()
    assert err <= 2 ** -8 * max(1e-3, ref.abs().max().item()) + 1e-6, (err, ref.abs().max().item())   # one bf16 rounding of the result
    pair = torch.zeros(rows, I, dtype=torch.bfloat16, device="cuda")
    T.tandem_test_gemm(T.BF16, 5, A, W, pair)                                                          # the CTA-pair launch of the same kernel
    assert torch.equal(pair, out)


def _nucleus(z, temperature, top_p, u, top_k=0):
    zt = torch.tensor(z, dtype=torch.float32, device="cuda")
    ut = torch.tensor(u, dtype=torch.float32, device="cuda")
    tok = torch.zeros(1, dtype=torch.int32, device="cuda")
    keep = torch.zeros(len(z), dtype=torch.uint8, device="cuda")
    T.tandem_test_nucleus(zt, temperature, top_p, ut, tok, keep, top_k=top_k)
    return int(tok.item()), keep.cpu().numpy().astype(bool)


def test_nucleus_hand_examples_and_ties():
    """The kept set of reading R10 on the hand example of tests/test_oracle_sampler.py, on exact ties (lower id first) and on a
    one-hot row; the expected masks come from oracle.sampler.kept_set_top_p."""
    from oracle.sampler import kept_set_top_p
    z = np.log(np.array([0.3, 0.05, 0.5, 0.15]))
    u = np.full(4, 0.5, dtype=np.float32)
    for top_p in (0.45, 0.51, 0.79, 0.81, 0.96, 1e-6):
        _, keep = _nucleus(z, 1.0, top_p, u)
        assert keep.tolist() == kept_set_top_p(z.astype(np.float32), 1.0, top_p).tolist(), top_p
    for V, top_p in ((4, 0.3), (4, 0.55), (7, 0.5), (1000, 0.25), (1000, 0.999)):      # all ids tie: a prefix by id
        _, keep = _nucleus(np.zeros(V), 1.0, top_p, np.full(V, 0.5, np.float32))
        want = kept_set_top_p(np.zeros(V, np.float32), 1.0, top_p)
        assert abs(int(keep.sum()) - int(want.sum())) <= (1 if abs(V * top_p - round(V * top_p)) < 1e-6 else 0) and keep[:keep.sum()].all()
    z = np.array([0., 2., 2., -1., 2., 2., 0.5]); u = np.full(7, 0.5, np.float32)        # four-way tie at the top
    for top_p in (0.1, 0.3, 0.5, 0.7):
        _, keep = _nucleus(z, 1.0, top_p, u)
        assert keep.tolist() == kept_set_top_p(z.astype(np.float32), 1.0, top_p).tolist(), top_p
    z = np.zeros(151936); z[77] = 1.0                                                     # a flat row: the threshold bin overflows the list
    for top_p in (0.3, 0.9):
        _, keep = _nucleus(z, 1.0, top_p, np.full(z.size, 0.5, np.float32))
        want = kept_set_top_p(z.astype(np.float32), 1.0, top_p)
        assert keep[77] and abs(int(keep.sum()) - int(want.sum())) <= 1 and keep[:keep.sum()].all()
    z = np.full(300, -30.0); z[123] = 10.0
    tok, keep = _nucleus(z, 0.7, 0.9, np.full(300, 0.5, np.float32))
    assert tok == 123 and keep.sum() == 1 and keep[123]


@pytest.mark.parametrize("V,temperature,top_p,seed", [(512, 0.7, 0.8, 0), (1000, 1.0, 0.5, 1), (4099, 0.6, 0.95, 2), (151936, 0.7, 0.8, 3),
                                                       (151936, 1.0, 0.2, 4)])
def test_nucleus_random_rows_match_oracle(V, temperature, top_p, seed):
    """Random rows (no exact ties): kept set identical to the oracle's float64 sort-and-cumsum except possibly the one id whose
    cumulative mass lands within fp32 rounding of top_p; sampled token identical."""
    from oracle.sampler import kept_set_top_p, sample_token
    rng = np.random.default_rng(seed)
    for rep in range(3):
        z = (rng.standard_normal(V) * 3.0).astype(np.float32)
        u = np.minimum((rng.integers(0, 1 << 32, size=V, dtype=np.uint64).astype(np.float32) + 0.5) * np.float32(2.0 ** -32),
                       np.float32(1 - 2.0 ** -24)).astype(np.float32)
        tok, keep = _nucleus(z, temperature, top_p, u)
        want = kept_set_top_p(z, temperature, top_p)
        assert int(np.sum(keep != want)) <= 1
        p = np.exp(z.astype(np.float64) / temperature); p /= p.sum()
        assert p[keep].sum() >= top_p - 1e-5 and (keep.sum() == 1 or p[keep].sum() - p[keep].min() < top_p + 1e-5)   # reaches top_p, minimal
        if np.array_equal(keep, want):
            assert tok == sample_token(z, temperature, top_p, u)


def test_top_k_hand_examples_ties_and_composition():
    """Reading R18 on the oracle's hand example, exact ties (lower id first), flat rows (the k-th largest sits in a bin that
    overflows the list), k = 1 = greedy, and top-k composed with top-p; masks from oracle.sampler.kept_set."""
    from oracle.sampler import kept_set
    z = np.log(np.array([0.3, 0.05, 0.5, 0.15]))
    u = np.full(4, 0.5, dtype=np.float32)
    for top_p, top_k in ((1.0, 1), (1.0, 2), (1.0, 3), (0.7, 3), (0.81, 2), (0.6, 2), (0.63, 2)):
        tok, keep = _nucleus(z, 1.0, top_p, u, top_k)
        assert keep.tolist() == kept_set(z.astype(np.float32), 1.0, top_p, top_k).tolist(), (top_p, top_k)
        if top_k == 1:
            assert tok == 2
    z = np.array([0., 2., 2., -1., 2., 2., 0.5]); u = np.full(7, 0.5, np.float32)
    for top_k in (1, 2, 3, 4, 5, 6):
        _, keep = _nucleus(z, 0.7, 1.0, u, top_k)
        assert keep.tolist() == kept_set(z.astype(np.float32), 0.7, 1.0, top_k).tolist(), top_k
    for V, top_k in ((1000, 20), (151936, 20), (151936, 2048), (5000, 1)):             # all ids tie: the first k ids
        _, keep = _nucleus(np.zeros(V), 1.0, 1.0, np.full(V, 0.5, np.float32), top_k)
        assert int(keep.sum()) == top_k and keep[:top_k].all()
    with pytest.raises(T.TandemError):                                                  # the list holds 2048 ids
        _nucleus(np.zeros(5000), 1.0, 1.0, np.full(5000, 0.5, np.float32), 3000)
    z = np.zeros(151936); z[[5, 100000, 77]] = [3.0, 2.0, 1.0]                          # three spikes on a flat row
    _, keep = _nucleus(z, 1.0, 1.0, np.full(z.size, 0.5, np.float32), 5)
    assert np.flatnonzero(keep).tolist() == [0, 1, 5, 77, 100000]


@pytest.mark.parametrize("V,temperature,top_p,top_k,seed", [(512, 0.7, 0.8, 20, 0), (1000, 1.0, 1.0, 50, 1), (4099, 0.6, 0.95, 7, 2),
                                                             (151936, 0.7, 0.8, 20, 3), (151936, 1.0, 1.0, 2048, 4), (151936, 0.7, 0.5, 1000, 5)])
def test_top_k_random_rows_match_oracle(V, temperature, top_p, top_k, seed):
    """Random rows: top-k is index work (bit-exact); with top-p on top the one id at the fp32 rounding boundary may differ."""
    from oracle.sampler import kept_set, sample_token
    rng = np.random.default_rng(seed)
    for rep in range(3):
        z = (rng.standard_normal(V) * 3.0).astype(np.float32)
        u = np.minimum((rng.integers(0, 1 << 32, size=V, dtype=np.uint64).astype(np.float32) + 0.5) * np.float32(2.0 ** -32),
                       np.float32(1 - 2.0 ** -24)).astype(np.float32)
        tok, keep = _nucleus(z, temperature, top_p, u, top_k)
        want = kept_set(z, temperature, top_p, top_k)
        if top_p >= 1.0:
            assert np.array_equal(keep, want) and int(keep.sum()) == top_k
        else:
            assert int(np.sum(keep != want)) <= 1 and not (keep & ~kept_set(z, temperature, 1.0, top_k)).any()
        if np.array_equal(keep, want):
            assert tok == sample_token(z, temperature, top_p, u, top_k)
