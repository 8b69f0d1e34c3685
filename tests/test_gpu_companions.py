"""GPU parity of the two companions of the attention path:
pf_rope and pf_kv_proj_grad vs their fp64 oracle definitions
(oracle/companions.py), through the C ABI."""
import numpy as np
import pytest
import torch

import oracle
from paper_2606_01143_b200 import binding as pf
from paper_2606_01143_b200 import inputs, schedule

pytestmark = pytest.mark.gpu

# one bf16 rounding of the output (2^-9 relative to the element, <= 2^-9 max|ref|) + fp32 sin/cos
ROPE_MAX_REL = 2.0 ** -8
# fp32 accumulation of L products of bf16 inputs against an fp64 sum: ~1e-7 sqrt(L) relative
GEMM_MAX_REL, GEMM_ABS = 2e-5, 1e-6


@pytest.fixture(scope="module")
def ctx():
    c = pf.pf_create(0)
    yield c
    pf.pf_destroy(c)


def _bf16(gen, *shape):
    return torch.randn(shape, generator=gen, dtype=torch.float32).to(torch.bfloat16)


def _positions(cu, pos0):
    return np.concatenate([pos0 + np.arange(cu[i + 1] - cu[i]) for i in range(len(cu) - 1)]) if len(cu) > 1 \
        else np.zeros(0, dtype=np.int64)


@pytest.mark.parametrize("H,d,cu,pos0", [
    (4, 128, [0, 300], 0),                       # the prefix: positions 0 .. Lp - 1
    (28, 128, [0, 129, 129, 193, 393], 5120),    # a packed suffix wave (one empty suffix), positions from Lp
    (8, 64, [0, 1, 65], 32768),                  # long prefix: the angle needs the fp64 reduction
    (2, 256, [0, 7], 1000003),
    (3, 16, list(range(0, 41)), 17),             # 40 one-token sequences: more than one launch of 32
])
@pytest.mark.parametrize("inverse", [False, True])
def test_rope_matches_oracle(ctx, H, d, cu, pos0, inverse):
    gen = torch.Generator().manual_seed(100 + d + pos0 % 97)
    x = _bf16(gen, cu[-1], H, d)
    ref = oracle.rope(x.to(torch.float64).numpy(), _positions(cu, pos0), 10000.0, inverse=inverse)
    y = x.cuda()
    pf.pf_rope(ctx, cu, pos0, y, 10000.0, inverse)
    got = y.cpu().to(torch.float64).numpy()
    assert np.isfinite(got).all()
    assert np.abs(got - ref).max() <= ROPE_MAX_REL * np.abs(ref).max()
    # per element: one bf16 rounding of the exact value (+ 1e-6 of fp32 sin/cos and products)
    assert (np.abs(got - ref) <= 2.0 ** -8 * np.abs(ref) + 1e-5 * np.abs(ref).max()).all()


def test_rope_positions_continue_across_the_seam(ctx):
    """RoPE of the suffix rows with pos0 = Lp is bit-identical to RoPE of the same rows
    inside the concatenated baseline sequence [P || S]; restarting at 0 is not."""
    gen = torch.Generator().manual_seed(7)
    Lp, Ls, H, d = 200, 77, 4, 128
    full = _bf16(gen, Lp + Ls, H, d).cuda()
    P, S, S0 = full[:Lp].clone(), full[Lp:].clone(), full[Lp:].clone()
    pf.pf_rope(ctx, [0, Lp + Ls], 0, full)
    pf.pf_rope(ctx, [0, Lp], 0, P)
    pf.pf_rope(ctx, [0, Ls], Lp, S)
    pf.pf_rope(ctx, [0, Ls], 0, S0)
    torch.cuda.synchronize()
    assert torch.equal(full[:Lp], P) and torch.equal(full[Lp:], S)
    assert not torch.equal(full[Lp:], S0)


def test_rope_strided_heads_in_place_and_inverse_round_trip(ctx):
    """A head slice of a fused QKV buffer is rotated in place (other heads untouched); the inverse
    brings it back to within two bf16 roundings."""
    gen = torch.Generator().manual_seed(9)
    L, H, d = 130, 6, 128
    buf = _bf16(gen, L, H, d).cuda()
    orig = buf.clone()
    view = buf[:, 2:5]
    pf.pf_rope(ctx, [0, L], 4096, view)
    torch.cuda.synchronize()
    assert torch.equal(buf[:, :2], orig[:, :2]) and torch.equal(buf[:, 5:], orig[:, 5:])
    assert not torch.equal(buf[:, 2:5], orig[:, 2:5])
    pf.pf_rope(ctx, [0, L], 4096, view, inverse=True)
    torch.cuda.synchronize()
    err = (buf.float() - orig.float()).abs().max().item()
    assert err <= 2 * 2.0 ** -8 * orig.float().abs().max().item()


def test_rope_error_paths(ctx):
    x = torch.zeros((8, 2, 128), dtype=torch.bfloat16, device="cuda")
    with pytest.raises(pf.PrefixFlowError):
        pf.pf_rope(ctx, [0, 8], 0, x[:, :, :24])                     # head_dim not a multiple of 16 / misaligned
    with pytest.raises(pf.PrefixFlowError):
        pf.pf_rope(ctx, [0, 8], -1, x)
    with pytest.raises(pf.PrefixFlowError):
        pf.pf_rope(ctx, [0, 8, 4], 0, x)                             # not monotone
    with pytest.raises(pf.PrefixFlowError):
        pf.pf_rope(ctx, [0, 8], 0, x, theta_base=1.0)
    pf.pf_rope(ctx, [0, 0], 0, x[:0])                                # empty: no-op


@pytest.mark.parametrize("L,dm,Hkv,d", [
    (1, 128, 1, 128),
    (333, 256, 4, 128),        # ragged last 64-token chunk
    (64, 128, 2, 64),          # 128 x 128 tile
    (200, 256, 1, 128),        # 256 x 128 tile
    (200, 384, 2, 128),        # 128 x 256 tile
    (5120, 3584, 4, 128),      # configs[1] prefix with a 7B-shaped d_model: 14 x 2 tiles of 256 x 256, split over tokens
    (777, 512, 8, 128),        # 256 x 256 tiles, 2 x 4 of them, ragged token range split 13 ways
])
def test_kv_proj_grad_matches_oracle(ctx, L, dm, Hkv, d):
    gen = torch.Generator().manual_seed(L + dm)
    X, dK = _bf16(gen, L, dm), _bf16(gen, L, Hkv, d)
    W0 = torch.randn((dm, Hkv * d), generator=gen, dtype=torch.float32)      # a pre-existing accumulator
    ref = W0.to(torch.float64).numpy() + oracle.kv_proj_grad(X.to(torch.float64).numpy(),
                                                              dK.to(torch.float64).numpy(), [], [])
    dW = W0.cuda()
    pf.pf_kv_proj_grad(ctx, X.cuda(), dK.cuda(), dW)
    got = dW.cpu().to(torch.float64).numpy()
    assert np.isfinite(got).all()
    assert np.abs(got - ref).max() <= GEMM_MAX_REL * np.abs(ref).max() + GEMM_ABS


def test_kv_proj_grad_strided_operands(ctx):
    """X as a column slice of a wider activation buffer, dY as the K part of a fused [L, 3, Hkv, d] buffer."""
    gen = torch.Generator().manual_seed(5)
    L, dm, Hkv, d = 200, 128, 2, 64
    Xw, qkv = _bf16(gen, L, dm + 64).cuda(), _bf16(gen, L, 3, Hkv, d).cuda()
    X, dK = Xw[:, 64:], qkv[:, 1]
    dW = torch.zeros((dm, Hkv * d), dtype=torch.float32, device="cuda")
    pf.pf_kv_proj_grad(ctx, X, dK, dW)
    ref = oracle.kv_proj_grad(X.cpu().to(torch.float64).numpy(), dK.cpu().to(torch.float64).numpy(), [], [])
    assert np.abs(dW.cpu().to(torch.float64).numpy() - ref).max() <= GEMM_MAX_REL * np.abs(ref).max() + GEMM_ABS


def test_dWk_split_over_the_three_phases(ctx):
    """PAPER.md:212 end to end on the GPU: run A -> B -> C, add the suffix terms X2(i)^T dK2(i) as
    Phase B produces them and the prefix term X1^T dK1 once after Phase C; the result equals the
    oracle's split formula fed with the oracle's own dK1 / dK2 (which the oracle pins tie to the sum
    over the N full-sequence replays)."""
    shape = inputs.small_case(4, 2, 64, 300, [129, 64, 200], seed=31, dist="unit")
    inp = inputs.make_group(shape)
    ref = oracle.group_reference(inp)
    gen = torch.Generator().manual_seed(3)
    dm = 128
    X1 = _bf16(gen, shape.Lp, dm)
    X2 = [_bf16(gen, L, dm) for L in shape.Ls]
    g = schedule.to_device(inp, wave=1)
    dW = torch.zeros((dm, shape.n_kv_heads * shape.head_dim), dtype=torch.float32, device="cuda")
    X2d = [x.cuda() for x in X2]
    schedule.run_prefixflow_step(ctx, g, after_each_suffix=lambda i: pf.pf_kv_proj_grad(ctx, X2d[i], g.dK2[i], dW))
    pf.pf_kv_proj_grad(ctx, X1.cuda(), g.dK1, dW)
    torch.cuda.synchronize()
    want = oracle.kv_proj_grad(X1.to(torch.float64).numpy(), ref.dK1,
                               [x.to(torch.float64).numpy() for x in X2], ref.dK2)
    got = dW.cpu().to(torch.float64).numpy()
    # dK1 / dK2 are bf16 outputs of the attention backward: the official gate of the path applies
    assert np.abs(got - want).max() <= 1e-2 * np.abs(want).max() + 1e-3
    rms = np.sqrt(((got - want) ** 2).sum() / (want ** 2).sum())
    assert rms <= 5e-3


def test_kv_proj_grad_error_paths(ctx):
    X = torch.zeros((64, 128), dtype=torch.bfloat16, device="cuda")
    dY = torch.zeros((64, 128), dtype=torch.bfloat16, device="cuda")
    dW = torch.zeros((128, 128), dtype=torch.float32, device="cuda")
    with pytest.raises(pf.PrefixFlowError):
        pf.pf_kv_proj_grad(ctx, X[:, :64], dY, dW[:64].contiguous())     # d_model not a multiple of 128
    with pytest.raises(pf.PrefixFlowError):
        pf.pf_kv_proj_grad(ctx, X, dY, dW[:, :64])                       # dW not contiguous / wrong shape
    with pytest.raises(pf.PrefixFlowError):
        pf.pf_kv_proj_grad(ctx, X[:32], dY, dW)                          # row counts differ
    pf.pf_kv_proj_grad(ctx, X[:0], dY[:0], dW)                           # L = 0: no-op
    torch.cuda.synchronize()
    assert float(dW.abs().max()) == 0.0


@pytest.mark.parametrize("L,dm,n_cols", [(130, 128, 128), (130, 256, 128), (130, 384, 256), (130, 256, 512)])
def test_kv_proj_grad_writes_only_dW(ctx, L, dm, n_cols):
    """dW sits between two guard bands of a known value: every tile variant's epilogue (one bulk
    reduce-add per accumulator row) stays inside the [d_model, n_cols] matrix."""
    gen = torch.Generator().manual_seed(11)
    X, dY = _bf16(gen, L, dm).cuda(), _bf16(gen, L, n_cols).cuda()
    guard = 1024
    arena = torch.full((guard + dm * n_cols + guard,), 7.0, dtype=torch.float32, device="cuda")
    dW = arena[guard:guard + dm * n_cols].view(dm, n_cols)
    dW.zero_()
    pf.pf_kv_proj_grad(ctx, X, dY, dW)
    torch.cuda.synchronize()
    assert bool((arena[:guard] == 7.0).all()) and bool((arena[guard + dm * n_cols:] == 7.0).all())
    ref = oracle.kv_proj_grad(X.cpu().to(torch.float64).numpy(), dY.cpu().to(torch.float64).numpy(), [], [])
    assert np.abs(dW.cpu().to(torch.float64).numpy() - ref).max() <= GEMM_MAX_REL * np.abs(ref).max() + GEMM_ABS
