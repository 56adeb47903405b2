"""CPU oracle for one confidence-thresholded denoising step of a masked diffusion LM.

TEST INFRASTRUCTURE ONLY.  Plain numpy float64, written from the paper
(/root/reference/PAPER.md, cited as P:<line>) and from the readings listed in DESIGN.md.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import it.  It shares no code with paper_2606_29094_b200/ (the CUDA path) and neither
imports the other.

Parity pins (tests/test_oracle_*.py, all `-m "not gpu"`):
  weights.py   closed-form moments of the Irwin-Hall(4) draw, hand-computed hash values
               for the splitmix64 finaliser (tests/golden/splitmix64.txt), bf16 RNE cases
  model.py     textbook softmax(QK^T/sqrt d)V by brute force; GQA == MHA with repeated K/V;
               RoPE norm preservation and position-shift invariance; zero-weight closed forms
  step.py      tau>1 => exactly one commit per step; tau<=0 => whole block per step; monotone
               progress; commits never change; F_cached(x;KV(x)) == F_full(x); L=1 cached
               trajectory == recompute-every-step trajectory; batch independence
  brute.py     scalar-loop twin (no matmul) agreeing with model.py/step.py on tiny shapes
  split-vocab  (max, sum-exp, argmax) merge == direct softmax for any tiling
  step.py      Step Predictor features (App. A, G22): library quantile on random data, hand cases, tau>1
               closed forms, frozen-at-commit, dry-run leaves the state alone
  sched.py     Alg. 1 / 4 / 5 (G18 readings): hand-worked numbers on a toy latency profile

parity unpinned: trained-model behaviour (Figure 2 example, "-38% steps at 0.7")
needs LLaDA/Dream weights and datasets that are not in this container.
"""
