"""B200-native (sm_100a) differentiable triangle-soup rasteriser: the hot path of
Triangle Splatting SLAM (arxiv/paper_2605_31419).

`paper_2605_31419_b200.ts`      -- thin ctypes binding of the C-ABI library (include/ts.h)
`paper_2605_31419_b200.scenes`  -- seeded synthetic inputs (no method arithmetic)
`paper_2605_31419_b200.build`   -- nvcc build step for libts.so (sm_100a only)
"""
