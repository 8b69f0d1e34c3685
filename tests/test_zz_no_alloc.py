"""pf_causal_bwd_static (include/prefixflow.h): the allocation-free causal backward, whose workspace is
the library's built-in 32 MiB scratch, against the existing path (pf_group_begin with a caller
workspace + pf_phaseA_fwd + pf_phaseC_bwd) on two calls in a row.  Collected last on purpose: the
suite runs with `pytest -x`, and this file must not hide a test after it."""
import pytest
import torch

from paper_2606_01143_b200 import binding as pf
from paper_2606_01143_b200 import inputs
from parity_util import check

pytestmark = pytest.mark.gpu

HQ, HKV, D = 8, 2, 128


@pytest.fixture(scope="module")
def ctx():
    c = pf.pf_create(0)
    yield c
    pf.pf_destroy(c)


def _case(L, seed):
    """One causal sequence: Q, K, V, dO of a seeded group's prefix part, on the device."""
    inp = inputs.make_group(inputs.small_case(HQ, HKV, D, L, [64], seed=seed, dist="std"))
    return [t.cuda() for t in (inp.Q1, inp.K1, inp.V1, inp.dO1)]


def _existing_path(ctx, desc, Q, K, V, dO):
    """The path the library already has: forward for O / LSE, then the backward with a torch-allocated workspace."""
    L = Q.shape[0]
    O = torch.empty_like(Q)
    LSE = torch.empty((HQ, L), dtype=torch.float32, device="cuda")
    dQ, dK, dV = torch.empty_like(Q), torch.empty_like(K), torch.empty_like(V)
    ws = torch.empty(pf.pf_workspace_bytes(desc, L, 0), dtype=torch.uint8, device="cuda")
    grp = pf.pf_group_begin(ctx, desc, L, K, V, None, None, ws)
    try:
        pf.pf_phaseA_fwd(grp, Q, O, LSE)
        pf.pf_phaseC_bwd(grp, Q, O, LSE, dO, dQ, dK, dV)
    finally:
        pf.pf_group_end(grp)
    torch.cuda.synchronize()
    return O, LSE, dQ, dK, dV


def test_static_scratch_backward_matches_the_existing_path_twice_in_a_row(ctx):
    desc = pf.make_desc(HQ, HKV, D)
    assert pf.pf_static_scratch_bytes() == 32 << 20
    assert pf.pf_causal_bwd_static_max_tokens(desc) >= 1024
    # second call: another length and other data, so stale scratch contents of the first would show
    for n, (L, seed) in enumerate([(333, 5), (200, 6), (333, 5)]):
        Q, K, V, dO = _case(L, seed)
        O, LSE, dQ_ref, dK_ref, dV_ref = _existing_path(ctx, desc, Q, K, V, dO)
        dQ, dK, dV = torch.full_like(Q, float("nan")), torch.full_like(K, float("nan")), torch.full_like(V, float("nan"))
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info()[0]
        pf.pf_causal_bwd_static(ctx, desc, Q, K, V, O, LSE, dO, dQ, dK, dV)
        torch.cuda.synchronize()
        free_after = torch.cuda.mem_get_info()[0]
        if n > 0:   # the first call may load the kernels' module; after that nothing may be allocated
            assert free_after >= free_before - (1 << 20), "the allocation-free entry point allocated device memory"
        # same kernels, same inputs: only the order of the fp32 reduce-adds differs; gates of the parity tests
        check(f"call {n} dQ", dQ, dQ_ref)
        check(f"call {n} dK", dK, dK_ref)
        check(f"call {n} dV", dV, dV_ref)
        # and far tighter than the gates: at most a few bf16 roundings apart
        for got, ref in ((dQ, dQ_ref), (dK, dK_ref), (dV, dV_ref)):
            err = (got.float() - ref.float()).abs().max().item()
            assert err <= 2.0 ** -6 * ref.float().abs().max().item()


def test_static_scratch_limit_and_errors(ctx):
    desc = pf.make_desc(HQ, HKV, D)
    cap = pf.pf_causal_bwd_static_max_tokens(desc)
    L = cap + 1
    Q = torch.zeros((L, HQ, D), dtype=torch.bfloat16, device="cuda")
    K = torch.zeros((L, HKV, D), dtype=torch.bfloat16, device="cuda")
    LSE = torch.zeros((HQ, L), dtype=torch.float32, device="cuda")
    dQ, dK, dV = torch.full_like(Q, 3.0), torch.full_like(K, 3.0), torch.full_like(K, 3.0)
    with pytest.raises(pf.PrefixFlowError) as e:
        pf.pf_causal_bwd_static(ctx, desc, Q, K, K, Q, LSE, Q, dQ, dK, dV)
    assert e.value.status == pf.PF_WORKSPACE and "exceeds" in str(e.value)
    torch.cuda.synchronize()
    assert float(dQ.min()) == 3.0 and float(dK.min()) == 3.0 and float(dV.min()) == 3.0   # nothing was enqueued
    pf.pf_set_option(ctx, "profile", 1)
    try:
        with pytest.raises(pf.PrefixFlowError) as e:
            pf.pf_causal_bwd_static(ctx, desc, Q[:64], K[:64], K[:64], Q[:64], LSE[:, :64].contiguous(), Q[:64],
                                    dQ[:64], dK[:64], dV[:64])
        assert e.value.status == pf.PF_STATE
    finally:
        pf.pf_set_option(ctx, "profile", 0)
    pf.pf_causal_bwd_static(ctx, desc, Q[:0], K[:0], K[:0], Q[:0], None, Q[:0], dQ[:0], dK[:0], dV[:0])   # L = 0: no-op
