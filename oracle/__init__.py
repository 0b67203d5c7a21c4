"""oracle/ -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

A plain, slow, obviously-correct CPU implementation of what the AnonShield hot path
(arxiv/paper_2606_15650, BASELINE.json north_star) computes.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import it.  It shares no code with ``paper_2606_15650_b200/`` and never imports it.

Modules
  encoder.py     numpy fp64 transformer-encoder NER forward + argmax
  decode.py      BIO span decode, window stitching, span byte gather
  crypto.py      ctypes front of anon_oracle.c: SHA-256, HMAC-SHA256,
                 cache dedup and pseudonym write-back

Pin status: every function is pinned by tests under
``tests/test_oracle_*.py`` except the paper's own example digits ``48624b5cdc`` (PAPER.md
L44), whose key is unpublished -- "parity unpinned" for that one literal only.
"""
