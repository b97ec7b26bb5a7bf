"""B200-native (sm_100a) hot path of RetroAttention (arxiv 2508.09001): one decode step of retrospective
sparse attention behind a C-ABI CUDA library.  See DESIGN.md.  `workload` (input generators) imports without
the CUDA extension; `binding` loads libretro.so and fails loudly if it is missing."""
