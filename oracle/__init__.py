"""CPU oracle for DARTS group-rollout decoding (arxiv/paper_2605_30859).

THIS PACKAGE IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may import it.  It shares no code with the CUDA path in
``paper_2605_30859_b200/`` and imports nothing from it; the CUDA path never
imports this package.

Everything is plain numpy in float64 (integers for the integer work), written
in the paper's order and notation so it can be checked against PAPER.md by eye.
Citations are ``PAPER.md:<line>`` plus the section / algorithm they fall in;
``DESIGN.md R<n>`` names a reading taken where the paper is silent or garbled.

Modules
-------
philox      Philox4x32-10 counter-based generator and the Gumbel noise built on it.
transformer Pre-norm GQA decoder (RMSNorm, RoPE, SwiGLU / top-k MoE): full causal
            forward (the definition) and incremental decode over a per-row KV list.
attention   softmax(q K^T / sqrt(hd)) V over [prefix || suffix] for one row (config 2).
sampling    temperature + Gumbel-max token choice with the top-2 margin.
selection   stop rules, the per-prompt DARTS rule (dual-end / shortest-only with
            proactive early stop, Alg. 2), active-set compaction.
rollout     lock-step group rollout (stepwise, with early stop) and the plain
            definition it must equal (roll everything out, then sort).

Parity pins (tests/test_oracle_*.py, run with -m "not gpu"):
  philox      Random123 known-answer vectors (tests/golden/philox4x32_10_kat.txt)
  gumbel-max  token histogram -> softmax(z/T) (chi-square); T=0 -> argmax
  attention   torch float64 scaled_dot_product_attention; rows sum to 1;
              prefix-shared == unshared; split-KV + LSE merge == unsplit
  rope        relative-position invariance;  rmsnorm  scale invariance / unit RMS
  transformer incremental decode == one full causal forward; == a torch library
              decoder with random norm weights (incl. the per-head QK-norm); zero
              weights -> uniform logits; MoE(E=1, top-1) == dense MLP; MoE(E
              identical experts, top-3) == dense MLP and scaled experts pin each
              gate to its own expert; qk_norm == torch rms_norm per head BEFORE rope
  selection   exhaustive enumeration on tiny pools vs. an independent brute-force
              statement of the rule; |sel| = K; EARLY == full-rollout-then-sort
  compaction  == stable partition
Trajectory *content* on random-init weights has no paper-printed value to pin
against (the paper prints no worked example of Alg. 2): "parity unpinned" beyond
the invariants above — see DESIGN.md.
"""

ACTIVE, VALID, TRUNC, PRUNED = 0, 1, 2, 3
MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP = 0, 1, 2
