// cao_gen_layout.h -- shared-memory layout of the fused generation kernel (host: cao_runs.cu, device: cao_gen_kernels.cuh).
#pragma once
#include <cstdint>

// Word offsets of the per-group shared-memory slice (computed on the host, cao_runs.cu: gen_layout()).
struct GenLayout {
    uint32_t rank, f, idx, x, v, pb, pbf, cand, key, scr, wl, cw, skey, bestrow;
    uint32_t words;                  // words per group (multiple of 4)
    uint32_t cta_words;              // CTA-wide prefix: probe target / pair lists (0 = read them from global memory)
    uint32_t G, NG;                  // threads per group, groups per CTA
};

#define GRP_SHARED_WORDS 16             // sizeof(GrpShared) / 4
