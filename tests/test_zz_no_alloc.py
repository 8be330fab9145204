"""GPU test (-m gpu) of lgx_eval_batch_static, the entry point for callers that cannot allocate device memory
when they call the library: a process that gave all free HBM to another owner at start-up (a framework's caching
allocator, a pre-sized cache), a loop with a latency bound that a stalling driver allocation would break, a plug-in
whose host forbids allocator calls after initialisation.  The call keeps its queue and counters in one fixed
16 MiB array inside the library's device image instead of taking them from the memory pool (include/lgx.h).

What is checked: on the same ids the new call's four outputs equal lgx_eval_batch's bit for bit (the bar of the
parity tests: flags equal, FP64 costs bit-equal), on TWO calls in a row — the second call finds the first one's
counters and queue records in the shared array and must clear what it needs; that a request above the stated
maximum is refused with LGX_ESTATIC and writes nothing; and that the maximum follows from the array's size.
The outputs are allocated by the test up front, as such a caller would do during its own set-up.

The file is named to be collected last (`pytest --collect-only`): `pytest -x` stops at the first failure, so
a failure here hides nothing.  It needs nothing from the tests before it and passes in a fresh process too."""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from paper_1909_10286_b200 import binding, workloads as wl


def _buffers(n, fill):
    dev = torch.device("cuda", torch.cuda.current_device())
    return (torch.full((n,), fill, dtype=torch.float64, device=dev), torch.full((n,), fill, dtype=torch.float64, device=dev),
            torch.full((n,), fill, dtype=torch.float64, device=dev), torch.full((n,), 7, dtype=torch.uint8, device=dev))


def _same(got, want, what):
    torch.cuda.synchronize()
    names = ("cost", "path_km", "makespan_h", "feasible")
    for k in (3, 0, 1, 2):
        a, b = got[k].cpu().numpy(), want[k].cpu().numpy()
        # view the doubles as integers: +inf rows and every finite bit pattern must agree exactly
        if a.dtype == np.float64:
            a, b = a.view(np.uint64), b.view(np.uint64)
        assert np.array_equal(a, b), f"{what}: {names[k]} differs from lgx_eval_batch"


@pytest.mark.parametrize("name", ["medium", "sweep"])
def test_static_scratch_matches_pooled_path_twice(name):
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the product path must fail loudly, not fall back")
    inst = wl.make(name)
    g = binding.Instance(inst)
    cap = g.eval_batch_static_max()
    rec = g.query(11)
    head = (64 + 16 * g.query(2) + 255) // 256 * 256
    assert cap == (binding.LGX_STATIC_SCRATCH_BYTES - head) // rec // 32 * 32 and cap >= 32
    # call 1: as many candidates as the array takes, implicit ids, ragged against the block size
    n1 = cap - 5
    want1 = g.eval_batch(inst.seed, first_id=3, n=n1)
    got1 = g.eval_batch_static(inst.seed, _buffers(n1, -1.0), first_id=3, n=n1)
    _same(got1, want1, f"{name}: first call")
    assert 0 < int(want1[3].sum()) < n1 or name == "sweep"       # both flag values on medium
    # call 2, straight after on the same stream: fewer candidates, explicit ids from the far end of the budget;
    # the array still holds call 1's counters and records
    n2 = max(cap // 3, 32) + 1
    ids = torch.from_numpy(wl.sample_ids(inst.budget, n2).astype(np.int64)).cuda()
    got2 = g.eval_batch_static(inst.seed, _buffers(n2, -2.0), ids=ids)
    want2 = g.eval_batch(inst.seed, ids=ids)
    _same(got2, want2, f"{name}: second call")
    # and the first request once more, after a different one has used the array
    got3 = g.eval_batch_static(inst.seed, _buffers(n1, -3.0), first_id=3, n=n1)
    _same(got3, want1, f"{name}: repeat of the first call")
    g.close()


def test_static_scratch_refuses_more_than_it_holds():
    if not torch.cuda.is_available():
        pytest.fail("no CUDA device: the product path must fail loudly, not fall back")
    inst = wl.make("medium")
    g = binding.Instance(inst)
    cap = g.eval_batch_static_max()
    out = _buffers(64, -4.0)
    launches = g.query(7)
    with pytest.raises(binding.LgxError) as ei:
        g.eval_batch_static(inst.seed, out, first_id=0, n=cap + 1)
    assert ei.value.code == binding.LGX_ESTATIC and "lgx_eval_batch_static_max" in str(ei.value)
    torch.cuda.synchronize()
    assert g.query(7) == launches                                   # refused before any launch
    assert float(out[0].max()) == -4.0 and int(out[3].min()) == 7   # and nothing written
    g.eval_batch_static(inst.seed, out, first_id=0, n=0)            # n = 0 is a no-op, as in lgx_eval_batch
    g.eval_batch_static(inst.seed, _buffers(cap, 0.0), first_id=0, n=cap)   # exactly the maximum is accepted
    torch.cuda.synchronize()
    g.close()
