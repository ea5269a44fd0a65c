"""Seeded random differential test of both attention kernels against the fp64 oracle: random supported shapes, random
mixes of decode rows / appended chunks / inert conversations, random prefix lengths around block, chunk (64-key) and
partition edges, random forced partition sizes, poisoned padding on or off.  Sizes stay small so the oracle takes seconds.
CSV_FUZZ_CASES raises the number of cases (default 24)."""
import os

import numpy as np
import pytest

from test_gpu_append import step_case

pytestmark = pytest.mark.gpu

SHAPES = [(32, 8, 128), (64, 8, 128), (4, 1, 64), (8, 8, 64), (16, 2, 128), (8, 8, 128), (8, 4, 128), (2, 1, 64), (16, 4, 64)]
EDGES = [0, 1, 15, 16, 17, 63, 64, 65, 127, 128, 129, 255, 256, 257, 1023, 1024, 1025, 2047, 2048, 2049]


def random_case(seed):
    rng = np.random.default_rng(1000 + seed)
    Hq, Hkv, d = SHAPES[int(rng.integers(0, len(SHAPES)))]
    n = int(rng.integers(1, 9))
    convs = []
    for _ in range(n):
        P = int(rng.choice(EDGES)) if rng.random() < 0.5 else int(rng.integers(0, 2600))
        kind = rng.random()
        if kind < 0.35:
            m = 1
        elif kind < 0.45:
            m = 0
        else:
            m = int(rng.choice([2, 3, 15, 16, 17, 31, 32, 33, 63, 64, 65, 100, 128, 129, 200])) if rng.random() < 0.7 \
                else int(rng.integers(2, 260))
        if m == 0 and P == 0:
            P = 5
        convs.append((P, m))
    if all(m == 0 for _, m in convs):
        convs[0] = (convs[0][0], 1)
    mpt = int(rng.choice([0, 0, 16, 64, 256, 1024]))
    return Hq, Hkv, d, convs, mpt, bool(rng.random() < 0.4), float(rng.choice([1.0, 1.0, 4.0])), float(rng.choice([0.0, 0.0, 1.0]))


@pytest.mark.parametrize("seed", range(int(os.environ.get("CSV_FUZZ_CASES", "24"))))
def test_random_tail_step_matches_the_oracle(oracle, seed):
    Hq, Hkv, d, convs, mpt, poison, qscale, v_mean = random_case(seed)
    step_case(oracle, 5000 + seed, Hq, Hkv, d, convs, mpt=mpt, poison=poison, v_mean=v_mean, qscale=qscale,
              what="fuzz %d %s %s mpt=%d poison=%s q x%g" % (seed, (Hq, Hkv, d), convs, mpt, poison, qscale))


@pytest.mark.parametrize("seed", range(int(os.environ.get("CSV_FUZZ_CASES", "24")) // 2))
def test_random_handoff_matches_the_oracle(oracle, seed):
    """kv_pack -> kv_unpack and kv_handoff_direct, single and batched: random layer counts, head counts, lengths and
    token offsets (ragged first and last blocks), random 16-bit patterns; whole pool image against the oracle's scatter."""
    from test_gpu_handoff import handoff_case

    rng = np.random.default_rng(9000 + seed)
    NL, Hkv, d = int(rng.integers(1, 4)), int(rng.choice([1, 2, 4, 8])), int(rng.choice([64, 128]))
    n = int(rng.integers(1, 40))
    convs = []
    for _ in range(n):
        tokens = int(rng.choice([1, 2, 15, 16, 17, 31, 32, 33])) if rng.random() < 0.5 else int(rng.integers(1, 200))
        convs.append((tokens, int(rng.integers(0, 40)) if rng.random() < 0.5 else 0))
    blocks = sum((o + t + 15) // 16 for t, o in convs) + int(rng.integers(1, 9))
    handoff_case(oracle, rng, NL, Hkv, d, blocks, convs, batched=bool(rng.random() < 0.6), direct=bool(rng.random() < 0.5))
