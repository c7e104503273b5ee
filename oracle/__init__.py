"""CPU oracle for the PersistentKV paged-decode hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2606_26666_b200/`` and neither imports the other.

* ``pkv_oracle.c`` / ``pkv_oracle.py`` -- FP64 attention through the block table (PAPER.md:39
  Eq. 1), split states and the exact merge.
* ``workqueue_oracle.py`` -- the split-bound policy and the compact workqueue as a pure-Python
  integer algorithm, plus the scheduler-derived counters of Table 4
  (PAPER.md:183-192).
* ``route_oracle.py`` -- the length-bucket route and the calibrated cost model
  with its gates and margins; the makespan form of its first term (A27).
* ``append_oracle.py`` -- the fused KV-append + RoPE step (PAPER.md:271 future work; A29).
* ``pkv_oracle.attention_fp8`` / ``attention_int8`` -- Eq. (1) on one-byte caches (A28).
"""
