"""cbm_trigger_select_noalloc: the list of selected events for callers that may not allocate device memory.

Who that is: a readout node that has handed out all of its device memory at start of run and must keep cudaMalloc /
cudaFree (which stall every stream of the device) out of its data-taking loop, or code that lives inside another
framework and only gets device pointers and a stream.  Every other entry point needs a handle, and creating a handle
allocates; this one keeps its scratch (the per-block counts of the compaction) in a fixed 16 KB array inside the
library image and therefore has a hard limit of K.NOALLOC_MAX_EVENTS events per call.

What is checked: the result is the same, element by element (index work: bit-exact, like every test of the list), as
the one of the existing path cbm_trigger_select_device on the same flags -- on two calls in a row, the second one
shorter than the first, so that whatever the first call left in the shared array would show up if the second call read
it.  The file sorts last on purpose (pytest -x stops at the first failure): it has to pass alone in a fresh process and
after all the other tests.
"""
import numpy as np
import pytest

from paper_1810_11966_b200 import workloads as W


def _flags(rng, n, p):
    a = (rng.random(n) < p).astype(np.uint8)
    a[a != 0] = rng.integers(1, 256, size=int(a.sum()), dtype=np.uint8)  # any non-zero byte means "accepted"
    return a


@pytest.mark.gpu
def test_select_noalloc_matches_select_device_on_two_calls_in_a_row():
    import torch
    from paper_1810_11966_b200 import binding as K
    rng = np.random.default_rng(20241106)
    cfg = W.CONFIGS[0]
    stream = torch.cuda.current_stream().cuda_stream
    # first call: 300 001 events = 74 blocks of 4096 and a ragged tail; second call: 4 097 events = 2 blocks, sparser flags
    calls = [(300_001, 0.4), (4_097, 0.03)]
    got = []
    for n, p in calls:  # the two no-allocation calls back to back, nothing else on the GPU in between
        a = _flags(rng, n, p)
        d_a = torch.from_numpy(a).cuda()
        d_ids = torch.full((n,), -1, dtype=torch.int32, device="cuda")
        d_n = torch.full((1,), -1, dtype=torch.int32, device="cuda")
        K.cbm_trigger_select_noalloc(n, d_a.data_ptr(), d_ids.data_ptr(), d_n.data_ptr(), stream)
        got.append((a, d_a, d_ids, d_n))
    torch.cuda.synchronize()
    with K.Trigger(cfg.layer_z, max(n for n, _ in calls), 16, n_slots=0) as trig:  # the existing path (allocates)
        for (n, _), (a, d_a, d_ids, d_n) in zip(calls, got):
            r_ids = torch.full((n,), -1, dtype=torch.int32, device="cuda")
            r_n = torch.full((1,), -1, dtype=torch.int32, device="cuda")
            trig.select_device(n, d_a, r_ids, r_n)
            torch.cuda.synchronize()
            count = int(r_n.item())
            assert count == int(np.count_nonzero(a)) and count > 0
            assert int(d_n.item()) == count
            # the whole output array: the ids, and the untouched fill value behind them
            assert torch.equal(d_ids, r_ids)
            assert np.array_equal(d_ids.cpu().numpy()[:count].view(np.uint32), np.flatnonzero(a).astype(np.uint32))


@pytest.mark.gpu
def test_select_noalloc_limit_empty_batch_and_null_pointers():
    import torch
    from paper_1810_11966_b200 import binding as K
    d_a = torch.ones(8, dtype=torch.uint8, device="cuda")
    d_ids = torch.full((8,), -1, dtype=torch.int32, device="cuda")
    d_n = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    # one event above the fixed limit: refused before anything is enqueued or read
    with pytest.raises(K.CbmTriggerError) as ei:
        K.cbm_trigger_select_noalloc(K.NOALLOC_MAX_EVENTS + 1, d_a.data_ptr(), d_ids.data_ptr(), d_n.data_ptr())
    assert ei.value.code == K.CBM_ERR_CAPACITY and "limit" in str(ei.value)
    with pytest.raises(K.CbmTriggerError) as ei:
        K.cbm_trigger_select_noalloc(8, d_a.data_ptr(), d_ids.data_ptr(), None)
    assert ei.value.code == K.CBM_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert int(d_n.item()) == -1 and bool((d_ids == -1).all())  # nothing was written by the refused calls
    # an empty batch writes the count only
    K.cbm_trigger_select_noalloc(0, None, None, d_n.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert int(d_n.item()) == 0
    # and the call still works after the refusals
    K.cbm_trigger_select_noalloc(8, d_a.data_ptr(), d_ids.data_ptr(), d_n.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    assert int(d_n.item()) == 8 and d_ids.cpu().tolist() == list(range(8))
