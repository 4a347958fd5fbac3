"""The replica merge's window / slice plan (paper_2606_24417_b200/replicas.py: merge_plan) as pure arithmetic, and the
peer-read exchange it drives emulated on numpy replicas: after reduce-scatter + all-gather every replica is the OR of
all.  (The gloo tests run the NCCL-shaped form with real processes; the GPU test runs this plan with the real kernels.)"""
import numpy as np
import pytest

from paper_2606_24417_b200 import replicas


@pytest.mark.parametrize("n,world,window", [(32 * 1000, 2, 32 * 64), (32 * 1001, 3, 32 * 100), (32 * 7, 8, 1 << 28), (32, 4, 64),
                                            (32 * 4096, 5, 40_000)])
def test_plan_covers_every_shard_exactly_once(n, world, window):
    plan = replicas.merge_plan(n, world, window)
    covered = np.zeros(n // 32, dtype=np.int32)
    prev_end = 0
    for a, slices in plan:
        assert a == prev_end and a % 32 == 0 and len(slices) == world
        pos = 0
        for lo, hi in slices:
            assert lo == pos and hi >= lo and lo % 32 == 0 and hi % 32 == 0
            covered[(a + lo) // 32:(a + hi) // 32] += 1
            pos = hi
        prev_end = a + pos
    assert prev_end == n and (covered == 1).all()


@pytest.mark.parametrize("world", [2, 3, 5])
def test_emulated_exchange_gives_the_or_of_all_replicas(world):
    rng = np.random.default_rng(world)
    n = 32 * 777
    reps = [rng.integers(0, 256, n, dtype=np.uint8) & rng.integers(0, 256, n, dtype=np.uint8) for _ in range(world)]
    want = np.bitwise_or.reduce(np.stack(reps), axis=0)
    for a, slices in replicas.merge_plan(n, world, 32 * 100):
        for j, (lo, hi) in enumerate(slices):                       # reduce-scatter by peer reads
            for p in range(world):
                if p != j:
                    reps[j][a + lo:a + hi] |= reps[p][a + lo:a + hi]
        for j, (lo, hi) in enumerate(slices):                       # all-gather
            for p in range(world):
                if p != j:
                    reps[p][a + lo:a + hi] = reps[j][a + lo:a + hi]
    for r in reps:
        assert np.array_equal(r, want)
