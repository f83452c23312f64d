"""B200-native BLINK imager hot path: gridding -> batched 2-D inverse FFT -> shift/normalise/real.

`paper_2405_13478_b200.blink` is the thin ctypes binding over the C-ABI library (include/blink.h);
`paper_2405_13478_b200.synth` holds the seeded synthetic workload generators (no method arithmetic);
`paper_2405_13478_b200.build` compiles csrc/ for sm_100a.  Nothing here imports oracle/.
"""
__version__ = "0.1.0"
