"""Small driver for ncu captures of the kernels bench.py does not put first (profiles/*.md name the commands):
  python -m paper_2606_01839_b200.profile_cases handoff   one kv_pack + kv_unpack + kv_handoff_direct of a 32-layer, 16384-token conversation
  python -m paper_2606_01839_b200.profile_cases tail      config 3 (agentic tail mix): paged_decode_attn + append_prefill_attn
Three calls each; inputs are the same seeded synthetic ones the tests and bench use."""
import sys

import numpy as np
import torch

from . import binding as B
from . import synth, workloads
what = sys.argv[1]
if what == "handoff":
    NL, Hkv, d, t = 32, 8, 128, 16384
    rng = np.random.default_rng(3)
    nb = synth.pool_blocks_for([t], slack=0.1)
    desc = B.pool_desc(NL, nb, Hkv, d)
    d_pool = torch.empty(B.kv_pool_bytes(desc) // 2, dtype=torch.int16, device="cuda")
    pool = B.KvPool(desc, d_pool); pool.set_free_order(synth.shuffled_free_order(rng, nb))
    k = torch.randint(-32768, 32767, (NL * t * Hkv * d,), dtype=torch.int16, device="cuda")
    v = torch.randint(-32768, 32767, (NL * t * Hkv * d,), dtype=torch.int16, device="cuda")
    st = torch.empty(B.kv_staging_bytes(desc, t) // 2, dtype=torch.int16, device="cuda")
    ids = torch.from_numpy(pool.alloc_blocks(synth.blocks_for(t))).cuda()
    for _ in range(3):
        B.kv_pack(desc, k, v, t, 0, st)
        B.kv_unpack(pool, st, t, 0, ids, len(ids))
        B.kv_handoff_direct(pool, k, v, t, 0, ids, len(ids))
    torch.cuda.synchronize()
else:
    wl = workloads.config_tail_workload(3)
    for _ in range(3):
        wl.decode(); wl.append()
    torch.cuda.synchronize()
print("ok")
