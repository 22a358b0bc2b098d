"""-m gpu: bgtq_block_energy_static -- the allocation-free entry point (scratch in a static device array of the library)
against the existing workspace path bgtq_block_energy, and against the oracle, on two calls in a row.

Collected last on purpose (the suite runs with pytest -x).  Passes alone in a fresh process and after the other tests:
it depends on nothing but the library and does not care what the static array held before.
"""
import numpy as np
import pytest

import workloads as W
from oracle import oracle as O

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def P():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_24033_b200 as pkg
    return pkg


def _inputs(seed, nq, nk, Hq, Hkv, dtype):
    scales = W.block_scales(seed, Hkv, 64)
    q = torch.from_numpy(W.pre_rope_gaussian(seed, 1, nq, Hq, 128, scales)).to(dtype).cuda()
    k = torch.from_numpy(W.pre_rope_gaussian(seed, 2, nk, Hkv, 128, scales)).to(dtype).cuda()
    return q, k


def _rel(a, b):
    a, b = a.double().cpu().numpy(), b.double().cpu().numpy()
    return float(np.max(np.abs(a - b) / np.maximum(np.abs(b), 1e-300)))


def test_static_scratch_entry_matches_workspace_path_twice_in_a_row(P):
    """Two calls back to back on the same stream, the second with a smaller, different problem (it would pick up the first
    call's leftovers if it read anything it had not written).  Bar: the block-energy bar of the other tests, rel 1e-5."""
    calls = [(101, 300, 70000, 16, 2, torch.float32, P.QK_AVG), (102, 64, 1000, 8, 4, torch.bfloat16, P.QK_PRODUCT)]
    outs = []
    ins = [_inputs(seed, nq, nk, Hq, Hkv, dt) for seed, nq, nk, Hq, Hkv, dt, _ in calls]
    bufs = [tuple(torch.full((c[4], 64), float("nan"), dtype=torch.float32, device="cuda") for _ in range(3)) for c in calls]
    torch.cuda.synchronize()
    held = torch.cuda.memory_allocated()
    for (q, k), (s, eq, ek), c in zip(ins, bufs, calls):            # no synchronisation between the two calls
        P.block_energy_static(q, k, s, kind=c[6], eq=eq, ek=ek)
    assert torch.cuda.memory_allocated() == held                    # the binding allocated nothing either
    torch.cuda.synchronize()
    for (q, k), (s, eq, ek), c in zip(ins, bufs, calls):
        s0, eq0, ek0 = P.block_energy(q, k, kind=c[6], return_parts=True)         # the existing path
        for got, ref in ((s, s0), (eq, eq0), (ek, ek0)):
            assert torch.isfinite(got).all()
            assert _rel(got, ref) <= 1e-5
        kind_name = {v: n for n, v in O.SCORE_KINDS.items()}[c[6]]
        so, eqo, eko = O.block_energy(q.double().cpu().numpy(), k.double().cpu().numpy(), kind=kind_name)
        for got, ref in ((s, so), (eq, eqo), (ek, eko)):
            assert np.max(np.abs(got.double().cpu().numpy() - ref) / ref) <= 1e-5
        outs.append(s.clone())
    # a third call repeating the first problem returns the first call's result bit for bit (deterministic, no state carried)
    s3 = torch.empty_like(bufs[0][0])
    P.block_energy_static(ins[0][0], ins[0][1], s3, kind=calls[0][6])
    torch.cuda.synchronize()
    assert torch.equal(s3, outs[0])


def test_static_scratch_entry_edge_cases_and_limit(P):
    lim = P.block_energy_static_max_row_elems()
    assert lim == 8192
    # keys only / queries only
    q, k = _inputs(103, 5, 77, 4, 4, torch.float32)
    s = torch.empty((4, 64), dtype=torch.float32, device="cuda")
    P.block_energy_static(q[:0], k, s, kind=P.K_ONLY)
    assert _rel(s, P.block_energy(q[:0], k, kind=P.K_ONLY)) <= 1e-5
    P.block_energy_static(q, k[:0], s, kind=P.Q_ONLY)
    assert _rel(s, P.block_energy(q, k[:0], kind=P.Q_ONLY)) <= 1e-5
    # exactly at the limit: 48 + 16 heads x 128
    q, k = _inputs(104, 40, 200, 48, 16, torch.bfloat16)
    s = torch.empty((16, 64), dtype=torch.float32, device="cuda")
    P.block_energy_static(q, k, s)
    assert _rel(s, P.block_energy(q, k)) <= 1e-5
    # beyond it: a clear error, nothing launched, the output untouched
    q, k = _inputs(105, 8, 8, 64, 8, torch.float32)
    s = torch.full((8, 64), -1.0, dtype=torch.float32, device="cuda")
    n0 = P.launch_count()
    with pytest.raises(P.BgtqError, match="static scratch limit"):
        P.block_energy_static(q, k, s)
    assert P.launch_count() == n0
    torch.cuda.synchronize()
    assert bool((s == -1.0).all())
