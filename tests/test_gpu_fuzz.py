"""Seeded fuzzing of the CUDA path against the oracle: random parameters (specialised and runtime-kernel
combinations), filter sizes that are not powers of two, ragged record batches of every length regime
(record mode, its device-side fallback, chunk mode), N runs, lower case, unaligned device pointers."""
import numpy as np
import pytest

import seqgen
from test_gpu_parity import check_parity, dev, gpu_query, sbf, oracle

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

PARAMS = [dict(k=31, m=16, s=28, H=4), dict(k=31, m=12, s=24, H=8), dict(k=31, m=20, s=31, H=1), dict(k=31, m=18, s=26, H=6),
          dict(k=31, m=14, s=30, H=2), dict(k=9, m=5, s=6, H=4), dict(k=32, m=16, s=28, H=4), dict(k=21, m=11, s=21, H=3),
          dict(k=15, m=15, s=12, H=5), dict(k=31, m=16, s=28, H=12), dict(k=25, m=9, s=20, H=4), dict(k=5, m=2, s=3, H=2)]


def _random_sequence(rng, n):
    seq = seqgen.uniform(int(rng.integers(1, 1 << 30)), n)
    for _ in range(int(rng.integers(0, 6))):                       # N runs of any length
        a = int(rng.integers(0, n)); seq[a:a + int(rng.integers(1, 400))] = ord("N")
    lower = rng.random(n) < 0.2
    seq[lower] |= 0x20
    if rng.random() < 0.5:                                          # a low-complexity stretch
        a = int(rng.integers(0, max(1, n - 3000))); seq[a:a + 3000] = np.frombuffer(b"ACAC" * 750, dtype=np.uint8)[:seq[a:a + 3000].size]
    return seq


def _random_offsets(rng, total):
    regime = int(rng.integers(0, 4))
    if regime == 0:
        return None                                                 # one sequence
    mean = [0, 60, 150, 5000][regime]
    lens = []
    left = total
    while left > 0:
        l = int(min(left, rng.integers(0, 2 * mean + 1)))
        if rng.random() < 0.03 and regime < 3:
            l = int(min(left, rng.integers(1500, 4000)))            # an occasional long record among short ones
        lens.append(l); left -= l
        if rng.random() < 0.05:
            lens.append(0)                                          # empty records
    return np.concatenate(([0], np.cumsum(lens))).astype(np.uint64)


@pytest.mark.parametrize("seed", range(24))
def test_fuzz_against_oracle(seed):
    rng = np.random.default_rng(1000 + seed)
    params = PARAMS[seed % len(PARAMS)]
    num_bits = int(rng.integers(1 << 10, 1 << 23))
    ins = _random_sequence(rng, int(rng.integers(40, 150_000)))
    q = _random_sequence(rng, int(rng.integers(1, 120_000)))
    m = min(q.size, ins.size) // 2
    q[:m] = ins[:m]                                                 # true members among the queries
    check_parity(params, num_bits, ins, _random_offsets(rng, ins.size), q, _random_offsets(rng, q.size))


def test_fuzz_unaligned_record_batches():
    rng = np.random.default_rng(77)
    ins = _random_sequence(rng, 90_001)
    o = oracle.OracleSBF(num_bits=1 << 20, k=31, m=16, s=28, H=4)
    o.insert_records(ins)
    with sbf.SuperBloomFilter(num_bits=1 << 20, k=31, m=16, s=28, H=4) as f:
        for shift in (1, 3, 7, 13):
            buf = dev(np.concatenate((np.zeros(shift, dtype=np.uint8), ins)))
            view = buf[shift:]
            assert view.data_ptr() % 16 == shift
            f.clear()
            sbf.sbf_insert_seq(f.handle, view.data_ptr(), ins.size)
            torch.cuda.synchronize()
            assert np.array_equal(f.export_bits(), o.export_bits())
            offs = _random_offsets(np.random.default_rng(shift), ins.size)
            bm = torch.full(((ins.size + 31) // 32,), -1, dtype=torch.int32, device="cuda")
            if offs is None:
                sbf.sbf_query_seq(f.handle, view.data_ptr(), ins.size, bm, None)
            else:
                sbf.sbf_query_records(f.handle, view.data_ptr(), dev(offs.view(np.int64)), offs.size - 1, ins.size, bm, None)
            torch.cuda.synchronize()
            want, _, _ = o.query_records(ins, offs)
            assert np.array_equal(bm.cpu().numpy().view(np.uint32), want)
    o.close()
