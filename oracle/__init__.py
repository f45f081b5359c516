"""CPU oracle for the CloakLM cloaked-layout hot path.  TEST INFRASTRUCTURE ONLY.

This package is a plain, slow, obviously-correct numpy restatement of what the hot path
computes (definitions O1-O12).  It exists so that the CUDA library
(`paper_2606_18400_b200/csrc`, C ABI in `include/cloak.h`) can be checked against something
that shares no code with it.

Rules this package keeps:
  * It imports nothing from `paper_2606_18400_b200` and the product imports nothing from it.
    Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs
    of `bench.py` may import it.
  * Integer work (Philox, tables, byte movement) is exact.  Floating point is evaluated in
    fp64 (inputs converted exactly, fp64 accumulation) and emitted as fp32 (O11, G17).
  * No blocking, fusion or reordering beyond what the cited definition states.
  * No input and no expected value ever comes from the CUDA path.

Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known answers + cuRAND host
generator; worked examples W1-W5 of SURVEY.md 8(c).4 under tests/golden/; O(n^2) brute-force
rank; bijection / restriction / forced-tie properties; byte-at-a-time restatement of O5;
unshuffle(shuffle)=id; relayout A->A = id, A->B->A; MLP' = MLP and attention' = attention
brute-forced in fp64; MoE' = MoE (expert + per-expert neuron permutation) brute-forced in fp64 with negative controls and
the E = 1 / k = 1 reductions to the dense MLP, and the stored eps / pi_e worked example of tests/golden/moe_example.json
(written by a pure-Python restatement that shares nothing with this package); attention closed forms (scale, causal mask,
grouped KV); adjacent_fraction against a python-int brute force on a table with descending neighbours; W = I and W = ones
closed forms for GEMV.  Parity unpinned: none.

Citations: `P:<n>` = /root/reference/PAPER.md line n; `BJ:` = BASELINE.json north_star /
configs; `O<n>`/`G<n>` = SURVEY.md section 8(c) definitions / readings.
"""
from .philox import philox4x32_10
from .keygen import (keygen, sort_pairs, STREAM_BLOCK, STREAM_PAGE, STREAM_TENSOR,
                     stream_mlp, stream_kvhead, stream_qgroup)
from .pool import (PoolGeometry, pool_geometry, PoolTables, pool_tables, shuffle_va,
                   shuffle_into, dump_view, unshuffle, relayout, rekey_pages, arena_plan,
                   adjacent_fraction, run_lengths, run_stats)
from .permute import (mlp_perm, head_maps, permute_mlp, permute_heads, expand_head_rows)
from .moe import (stream_expert, stream_expert_mlp, expert_perm, expert_mlp_perm, permute_experts,
                  topk_experts, moe_f64)
from .linear import (to_f64, f32_to_bf16_bits, bf16_bits_to_f32, linear_f64, mlp_f64,
                     attention_f64, to_tile128, from_tile128, err_normwise,
                     err_elementwise_floored)
