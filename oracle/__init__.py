"""CPU fp64 oracle for the STAR-KV latent-cache hot path.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with the CUDA path
(``paper_2606_08382_b200``): neither imports the other, and both are written from the paper
(/root/reference/PAPER.md, cited as ``PAPER.md:L<line>``) and from the cache-format text in
DESIGN.md ("Cache page format v1").

What each module computes and the passage it follows:

``layout``     byte map of one cache page (DESIGN.md format v1; not in the paper: PagedAttention
               is only cited).
``codec``      low-rank-aware mixed-precision per-token quantiser, §4.4,
               Eq.12 L208 (leading channels at b_out, trailing at b_in, per-token), and the
               pack/unpack of latents into pages.
``attention``  decode attention by the plain definition: dequantise, reconstruct
               K = K' U_K^T and V = V' U_V^T (§3.2), textbook softmax attention
               (§3.1) with GQA head mapping; plus an independent absorbed-form
               path (§3.3) used only for identity tests.
``append``     compress-on-append: K' = x (Sigma V)_K per head, V' = x (Sigma V)_V joint
               (§3.2), round to fp16, quantise (Eq.12), write into pages.
``analysis``   factor construction by truncated SVD (L58), hard threshold (Eq.1), JD/HD
               approximations (Lemma 4.1/4.2 L155-184), bit/compression and FLOP accounting
               (Table 4, Table 11), block Hadamard
               fusion (L206-210).

Pins (tests/test_oracle_*.py, ``-m "not gpu"``) are listed in DESIGN.md "Oracle pins".
Parity unpinned (stated here as required): agreement with the authors' own quantiser details
(symmetric absmax, RNE, fp16 scale, 20% split rounding: DESIGN.md readings A5, A8, A11), their
cache layout, and their treatment of uncompressed layers 0/1/31 (A19) -- the paper gives no
worked numeric example for any of these.
"""
