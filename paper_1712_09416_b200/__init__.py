"""B200-native (sm_100a) ALICE HLT TPC sector tracker hot path (arxiv 1712.09416): CA neighbour finding,
link cleaning, start hits, Kalman-filter tracklet construction, tracklet selection -- behind the C ABI of
``include/tpctrack.h``.

* ``paper_1712_09416_b200.tracker`` -- thin ctypes binding of ``csrc/libtpctrack.so`` (argument marshalling
  only; fails loudly when the CUDA library is missing -- there is no CPU fallback).
* ``paper_1712_09416_b200.gen``     -- seeded synthetic events (inputs only; none of the method's arithmetic).
"""

__all__ = ["tracker", "gen"]
