"""cap_dispatch_layout_static -- the S5 entry point that allocates nothing (static device scratch of
CAP_STATIC_SCRATCH_BYTES inside the library) -- against the existing cap_dispatch_layout path (caller
workspace) and the CPU oracle: bit-exact, on two calls in a row that share the scratch array (the second
one smaller, so stale contents of the first would show), plus the size limit.  Collected last on purpose
(the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu

from oracle import cap_oracle as O                      # noqa: E402
from paper_2607_05116_b200 import cap                   # noqa: E402
from parity_util import dev, host                       # noqa: E402


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    cap.lib()


def _case(rng, T, k, E, D, masked):
    idx = np.stack([rng.permutation(E)[:k] for _ in range(T)]).astype(np.int32)
    pi = rng.integers(0, D, E).astype(np.int32)
    pi[rng.integers(0, E)] = D - 1
    kept = (rng.random((T, k)) < 0.6).astype(np.uint8) if masked else None
    return idx, pi, kept


def _run_both(idx, pi, kept, D):
    T, k = idx.shape
    idx_d, pi_d, kept_d = dev(idx), dev(pi), dev(kept)
    # outputs owned by the caller, filled with a poison value first
    sp = torch.full((T * k,), -7, dtype=torch.int32, device="cuda")
    pos = torch.full((T * k,), -7, dtype=torch.int32, device="cuda")
    off = torch.full((D + 1,), -7, dtype=torch.int64, device="cuda")
    n0 = cap.launch_count()
    cap.dispatch_layout_static(idx_d, kept_d, pi_d, D, sp, off, pos)
    torch.cuda.synchronize()
    assert cap.launch_count() - n0 == 3                                   # the same three kernels
    sp_e, off_e, pos_e = cap.dispatch_layout(idx_d, kept_d, pi_d, D)      # existing path, caller workspace
    torch.cuda.synchronize()
    n = int(off_e[-1])
    assert torch.equal(off, off_e)
    assert torch.equal(sp[:n], sp_e[:n])
    assert torch.equal(pos, pos_e)
    sp_r, off_r, pos_r = O.dispatch_layout(idx, pi, D, kept=kept)         # and the oracle
    assert np.array_equal(host(off), off_r) and np.array_equal(host(sp)[:n], sp_r) and np.array_equal(host(pos), pos_r)


def test_static_scratch_two_calls_in_a_row_match_the_workspace_path():
    assert cap.lib().cap_static_scratch_bytes() == 4 * 1024 * 1024
    rng = np.random.default_rng(20260705)
    # first call: config-3 shape (65 536 tokens, top-8, 16 destinations), pruned trace
    _run_both(*_case(rng, 65536, 8, 128, 16, True), 16)
    # second call right behind it on the same array: smaller, other D, ragged tail, unpruned
    _run_both(*_case(rng, 4099, 10, 512, 64, False), 64)
    # and a third that grows again
    _run_both(*_case(rng, 30001, 3, 64, 5, True), 5)


def test_static_scratch_limit_and_empty():
    E, k, D = 512, 10, 64
    need = lambda T: int(cap.lib().cap_workspace_bytes(cap.CALL_DISPATCH_LAYOUT, 1, T, E, k, D, 0))
    limit = int(cap.lib().cap_static_scratch_bytes())
    T_big = 1 << 20
    assert need(T_big) > limit
    idx = torch.zeros((T_big, k), dtype=torch.int32, device="cuda")
    pi = torch.zeros((E,), dtype=torch.int32, device="cuda")
    sp = torch.empty((T_big * k,), dtype=torch.int32, device="cuda")
    off = torch.full((D + 1,), -7, dtype=torch.int64, device="cuda")
    n0 = cap.launch_count()
    with pytest.raises(cap.CapError, match="EWORKSPACE.*static array holds"):
        cap.dispatch_layout_static(idx, None, pi, D, sp, off)
    torch.cuda.synchronize()
    assert cap.launch_count() == n0 and int(off[0]) == -7                 # refused before any launch
    # the largest T that still fits is served
    T_fit = max(t for t in (1 << 17, 1 << 16) if need(t) <= limit)
    rng = np.random.default_rng(3)
    i2, p2, k2 = _case(rng, 2048, k, E, D, True)
    reps = T_fit // 2048
    _run_both(np.tile(i2, (reps, 1)), p2, np.tile(k2, (reps, 1)), D)
    # T = 0: offsets zeroed, nothing else touched
    cap.dispatch_layout_static(idx[:0], None, pi, D, sp, off)
    torch.cuda.synchronize()
    assert host(off).tolist() == [0] * (D + 1)
