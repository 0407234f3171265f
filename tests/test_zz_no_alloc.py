"""`-m gpu`, collected last on purpose: fire_fitness_static, the entry point that allocates nothing (include/fire.h).

Its scratch (the per-simulation counts of Eq. 2 and #A) is a static device array inside the library instead of a buffer the handle
allocates.  The check is against the existing path, fire_fitness, on the same inputs: scores bit for bit (the tolerance the other
fitness tests use) and the same reference area, on two calls in a row whose second batch is smaller and different, so that counts
left in the array by the first call would show.  Runs alone in a fresh process and after the other tests alike: it makes its own
inputs and touches no state of theirs."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")
if not torch.cuda.is_available():                       # collected on the CPU box too; never runs there
    pytest.skip("needs a CUDA device", allow_module_level=True)


def _maps(rng, S, H, W):
    Ww = (W + 31) // 32
    mask = np.zeros((Ww * 32,), bool); mask[:W] = True
    tail = np.packbits(mask, bitorder="little").view("<u4")
    ref = rng.integers(0, 2 ** 32, (H, Ww), dtype=np.uint32) & tail
    burned = rng.integers(0, 2 ** 32, (S, H, Ww), dtype=np.uint32) & tail
    burned[0] = ref
    if S > 1:
        burned[1] = 0
    return ref, burned


def test_fitness_static_equals_fire_fitness_on_two_calls_in_a_row():
    import gpu_helpers as gh
    from paper_1701_03549_b200 import libfire as lf

    rng = np.random.default_rng(20260101)
    H, W = 130, 203                                              # ragged width, rows of 7 words (scalar path of the counting kernel)
    ls = {"veg": rng.integers(1, 4, (H, W)).astype(np.uint8), "slope": np.zeros((H, W), np.float32),
          "aspect": np.zeros((H, W), np.float32), "wind": np.zeros((H, W), np.float32)}
    L = gh.make_landscape(ls)                                    # the existing path needs a handle; the new one does not
    calls = [(300, 0), (41, 1)]                                  # (S, metric): the second batch is smaller, other maps, other metric
    inputs = []
    for S, metric in calls:
        ref, burned = _maps(rng, S, H, W)
        inputs.append((gh.dev(ref), gh.dev(burned), torch.empty((S,), dtype=torch.float32, device="cuda"),
                       torch.full((1,), -1, dtype=torch.int32, device="cuda"), ref, burned, metric))
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    for ref_d, burned_d, score, area, _, _, metric in inputs:     # two calls in a row on one stream, nothing in between
        lf.fire_fitness_static(ref_d, burned_d, W, metric, score, area)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] >= free_before           # nothing was allocated on the device by those calls
    for ref_d, burned_d, score, area, ref, burned, metric in inputs:
        counts, want, N = gh.fitness(L, ref, burned_d, metric)
        got = score.cpu().numpy()
        assert np.array_equal(got.view(np.uint32), want.view(np.uint32))                       # bit-exact floats
        assert int(area.cpu().numpy().view(np.uint32)[0]) == N == int(np.unpackbits(ref.view(np.uint8)).sum())
    # a 16 B aligned shape (vector path), at the largest batch the array holds, then one simulation more: a clear error
    H2, W2 = 8, 128
    S2 = lf.FIRE_FITNESS_STATIC_MAX_SIMS
    ref, burned = _maps(rng, S2 + 1, H2, W2)
    L2 = gh.make_landscape({k: v[:H2, :W2].copy() for k, v in ls.items()})
    ref_d, burned_d = gh.dev(ref), gh.dev(burned)
    score = torch.empty((S2,), dtype=torch.float32, device="cuda")
    lf.fire_fitness_static(ref_d, burned_d[:S2], W2, 0, score)
    torch.cuda.synchronize()
    _, want, _ = gh.fitness(L2, ref, burned_d[:S2], 0)
    assert np.array_equal(score.cpu().numpy().view(np.uint32), want.view(np.uint32))
    with pytest.raises(lf.FireError) as err:
        lf.fire_fitness_static(ref_d, burned_d, W2, 0, torch.empty((S2 + 1,), dtype=torch.float32, device="cuda"))
    assert err.value.code == lf.FIRE_ELIMIT and "limit" in str(err.value)
    # the rejected call enqueued nothing and the array still works
    lf.fire_fitness_static(ref_d, burned_d[:5], W2, 1, score[:5])
    torch.cuda.synchronize()
    _, want, _ = gh.fitness(L2, ref, burned_d[:5], 1)
    assert np.array_equal(score[:5].cpu().numpy().view(np.uint32), want.view(np.uint32))
    L.close(); L2.close()
