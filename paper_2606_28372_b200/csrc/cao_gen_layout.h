// cao_gen_layout.h -- shared-memory layout of the fused generation kernel (host: cao_runs.cu, device: cao_gen_kernels.cuh).
#pragma once
#include <cstdint>

// Word offsets of the per-group shared-memory slice (computed on the host, cao_runs.cu: gen_layout()).
struct GenLayout {
    uint32_t rank, f, idx, x, v, pb, pbf, cand, key, scr, wl, cw, skey, bestrow, Lc, aux4, ptab;
    uint32_t words;                  // words per group (multiple of 4)
    uint32_t cta_words;              // CTA-wide prefix: strides, upper coordinates, Hamming-1 neighbour list, probe lists
    uint32_t NB, nb_words;           // Hamming-1 neighbours of a point = sum (m_d - 1); words of their list
    uint32_t probe_in_smem;          // the target / pair lists of the Hamming-2/3 probe are copied to shared memory
    uint32_t G, NG;                  // threads per group (a multiple of roundup32(P): groups are widened while the GPU is underfilled), groups per CTA
    uint32_t wide;                   // Firefly: four adjacent lanes share one firefly (G = 4 * roundup32(P))
};

#define GRP_SHARED_WORDS 48             // sizeof(GrpShared) / 4
