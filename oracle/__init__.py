"""fp64 CPU oracle for the MURMUR intra-chunk hot path (arxiv/paper_2606_01483).

TEST INFRASTRUCTURE ONLY.  Nothing under ``oracle/`` is part of the product: only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import, call, link or execute it.  It shares no code with the CUDA
path in ``paper_2606_01483_b200/`` (no common kernels, headers, helpers or constants) and
neither imports the other; only the seeded input generators in ``workloads/`` serve both.

What it computes (PAPER.md = /root/reference/PAPER.md):

* ``policy``       - the retained ("attended") set A(t) and resident set R(t) of the hybrid
                     sliding-window policy: Alg. 1 on the output region,
                     Eq. 2 / Alg. 2 on the speech region, system prompts
                     always kept.  Closed form, evaluated per position.
* ``literal_sim``  - Alg. 1 and Alg. 2 transcribed line by line as loops over decode steps
                     keeping Python sets; an independent second implementation of A(t)/R(t).
* ``paged_cache``  - plain-integer simulation of the paged cache bookkeeping the policy
                     implies (position-paged blocks, deterministic LIFO free stack,
                     compacted live-page list, run descriptors).  DESIGN.md readings C2/C3.
* ``attention``    - Eq. 1: exact max-subtracted softmax attention over
                     the retained set in fp64, GQA head map h -> h // G, and the
                     log-sum-exp merge of partial results.
* ``sparsity``     - the attention-sparsity profile of PAPER.md:77 / Fig. 5: the
                     fewest tokens holding 99 % of a head's attention mass, split by region, and
                     the mass a candidate window policy preserves.
* ``prefill``      - causal self-attention of the prefill tokens: Eq. 1 of each
                     prefill position over the positions up to and including itself.
* ``indexset``     - general index-set eviction (the future work of PAPER.md:224): per-(layer, KV head) retained
                     index sets, dense stable compaction, head-ragged append, Eq. 1 over the slabs, and the
                     mass-set producer of query-aware sets.  A convention of this build: parity unpinned
                     against the paper, pinned against its defining properties.
* ``cost_model``   - Eq. 3 theoretical attention-cost ratio.
* ``c/``           - a plain C twin of ``attention`` (fp64, optional OpenMP) used for the
                     timed CPU baseline; checked against ``attention`` in tests.

Parity status: every function here is pinned by ``tests/test_oracle_*.py`` (run with
``-m "not gpu"``) against values the paper prints, closed forms, brute force on tiny
inputs and library routines.  Conventions that the paper does not fix (page-id order,
default d/k_o/k_s) are listed as "convention, not pinned by the paper" in DESIGN.md.
"""
