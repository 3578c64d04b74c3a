"""CPU float64 oracle for the Aframe streaming detection statistic (arXiv 2403.18661).

TEST INFRASTRUCTURE ONLY.  Plain, slow, obviously-correct numpy float64 restatement of
what the hot path computes, written from /root/reference/PAPER.md (cited as P:<line>)
and the readings of SURVEY.md 8(c) / DESIGN.md (tags A1..C3).  It shares no code with
the CUDA path (paper_2403_18661_b200/csrc) and neither imports the other.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl
reference`` legs may import it; the product path never does.

Modules
-------
fft      naive O(N^2) DFT (the definition), own radix-2 FFT, real transforms
psd      O-1  Welch PSD ("estimate the PSD"; reading A1, A2)
whiten   O-2  whitening-filter design, O-3 FIR whitening (A3-A6)
network  O-5  1D ResNet forward from the layer table (B1-B8)
stream   O-4  window unfold, O-6 streaming / rolling-PSD rule, timeslides
postprocess  NEXT-1  1 s top-hat integration of the scores, 8 s clustering -> triggers (readings D1-D3)

Parity pins: every function above is pinned in tests/test_oracle_*.py against a closed
form, a library routine (numpy.fft, scipy.signal.welch, scipy.signal.lfilter/torch conv)
or brute force.  Functions whose *convention* the paper does not fix are listed as
"parity unpinned by the paper" in DESIGN.md (readings A7, B2, C2): the arithmetic is
pinned, the choice of convention is not.
"""
