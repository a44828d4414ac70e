"""fp64 CPU oracle for the SpotAttention hot path (arxiv/paper_2606_22874).

THIS PACKAGE IS TEST INFRASTRUCTURE.  It is a plain, slow, obviously-correct
restatement of what /root/reference/PAPER.md defines, written in numpy fp64
(pure-Python loops for the brute-force pins).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import it.  The product
(``paper_2606_22874_b200``) never imports it, shares no code, table or constant
generator with it, and has no CPU fallback.

Modules (each function cites the PAPER.md passage it restates):

* ``bf16``       - exact BF16-bits -> float64 decode (inputs are BF16 bit
                   patterns; the oracle computes in fp64 on the exact values).
* ``quant``      - step a0: the two group-32 selector-K quantisers and their
                   dequantisers (readings R16/R17).
* ``selection``  - steps a1/a2: selector score, per-block max
                   (PAPER.md:71), static top-K (Eq. 6), dual top-p
                   with reserved sink/recency tier and K_min floor (Eq. 7-8,
                   PAPER.md:83-92), decode form and query-block (prefill) form.
* ``attention``  - steps a3/a3': softmax attention over the tokens of the
                   selected blocks (PAPER.md:47 Fig. 2, :71), GQA, decode form
                   and causal chunked-prefill form; a second, independent
                   mask-form coding; plain dense attention.
* ``projection`` - upstream step f1: selector projections W_q h, W_k h, W_w h and
                   the rotary embedding of q^I / k^I (
                   DESIGN.md readings R27-R29).
* ``training``   - f4: the training-side reductions -- head-averaged teacher
                   distribution (Eq. 1), student softmax (Eq. 2), DenseKL (Eq. 3)
                   and SparseKL renormalised on the selector's own top-K set
                   (Eq. 4); readings R34-R36.
* ``brute``      - exhaustive enumeration used to pin the nucleus rule on tiny
                   inputs.

Parity pins (tests/test_oracle_*.py, ``-m "not gpu"``) and which functions
remain "parity unpinned" are listed in DESIGN.md section 4.

PARITY UNPINNED: ``selection.tile_scores_prefill`` -- the paper does not say
how a query *block* reduces to one tile score ("one score per
query-block x key-block tile"); reading R2 takes the max over the
block's queries.  It is pinned only through its reduction to the decode form at
q_block = 1 and the bound "tile score >= every member query's block score".
"""
