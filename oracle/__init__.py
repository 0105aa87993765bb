"""CPU oracle for the coalesced-chunk hot path of TurboServe (arxiv/paper_2606_19271).

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and the
`cpu_baseline` / `--impl reference` legs of `bench.py` may import this package.  The
product path (`paper_2606_19271_b200/`) never imports it, and this package never
imports the product path: the two share no code.  Only `synth/` (seeded input
generators, no arithmetic of the method) serves both.

What it computes follows PAPER.md §3.1 (:66 coalesced chunk execution, :74 session
lifecycle, :76 GPU-CPU offloading) and §6.1 (:261 isolated per-session state regions,
ownership table), with every numerical detail the paper leaves open taken from
BASELINE.json `north_star` / SURVEY.md §8(c) readings R1-R18 (listed in DESIGN.md).
Plain numpy, fp64 arithmetic, no blocking/fusion/online tricks.

Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 brute force, P2 constant V, P3 single
visible key, P4 placement invariance, P5 suspend/resume identity, P6 reduction to
torch SDPA, P7 chunked == monolithic, P8 batch-composition invariance, P9 softmax
invariants + LSE merge, P10 window equivalence + page-count closed forms, P11
hand-worked allocator trace (tests/golden/tiny_allocator_trace.txt), P12 distribution
sanity, P13 `attention_rows` (the sampled-row entry point of the full-size parity tests and
of bench.py's cpu_baseline) against `chunk_attention` on a rolled-window multi-head pool
and against explicit loops over the logical arrays, P14 the bf16 conversions (`_widen`,
synth.bf16) against torch.bfloat16 on all 65 536 patterns / 1.4 M fp32 values incl. ties;
migration (O4, `OraclePool.migrate_to`): M1 hand-worked id trace
(tests/golden/migration_trace.txt), M2 == suspend + transplant + resume, M3 round trip and
attention invariance, M4 conservation.  Parity unpinned: none.
"""
from .pool import OraclePool, OracleError, INVALID, STATE, NO_PAGES, NO_HOST, CAPACITY, RESIDENT, SUSPENDED
from .attention import chunk_attention, attention_rows
from .scheduler import SchedulerOracle

__all__ = ["OraclePool", "OracleError", "INVALID", "STATE", "NO_PAGES", "NO_HOST", "CAPACITY",
           "RESIDENT", "SUSPENDED", "chunk_attention", "attention_rows", "SchedulerOracle"]
