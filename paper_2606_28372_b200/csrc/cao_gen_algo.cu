// cao_gen_algo.cu -- instantiates the fused generation kernel (cao_gen_kernels.cuh) for ONE algorithm.  The build
// compiles this file four times (-DCAO_GEN_ALGO=0..3: DE, PSO, Firefly, GA) into separate objects, in parallel.
#include "cao_gen_kernels.cuh"

#ifndef CAO_GEN_ALGO
#error "compile with -DCAO_GEN_ALGO=0..3"
#endif
#define CAO_CAT_(a, b) a##b
#define CAO_CAT(a, b) CAO_CAT_(a, b)

// Opt-in shared memory (always the device maximum, see cao_smem_optin_max: run sets that share an instantiation must not
// lower the limit under one another) + resident CTAs per SM of the variant that (roww, threads) selects.
int CAO_CAT(cao_gen_setup_, CAO_GEN_ALGO)(int roww, unsigned threads, size_t smem, int wide, int* occ) {
#define SETUP(W, T)                                                                                                        \
    do {                                                                                                                   \
        CAO_SMEM_OPTIN((k_gen<CAO_GEN_ALGO, W, T>));                                                                       \
        CAO_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, k_gen<CAO_GEN_ALGO, W, T>, (int)threads, smem));       \
    } while (0)
#if CAO_GEN_ALGO == 2
    if (wide && roww == 4 && threads <= 256) {                         // Firefly, four lanes per firefly: its own instantiation
        CAO_SMEM_OPTIN((k_gen<2, 4, 256, true>));
        CAO_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ, k_gen<2, 4, 256, true>, (int)threads, smem));
        return CAO_OK;
    }
#endif
    (void)wide;
    if (roww == 4) { if (threads <= 256) SETUP(4, 256); else SETUP(4, 1024); }
    else           { if (threads <= 256) SETUP(8, 256); else SETUP(8, 1024); }
#undef SETUP
    return CAO_OK;
}

int CAO_CAT(cao_gen_launch_, CAO_GEN_ALGO)(int roww, unsigned grid, unsigned threads, size_t smem, cudaStream_t st,
                                           const SpaceMeta& sm, const ProbeMeta& pm, const RunsMeta& rm, const GenLayout& lay,
                                           uint32_t g_first, uint32_t n_gens) {
#define LAUNCH(W, T) k_gen<CAO_GEN_ALGO, W, T><<<grid, threads, smem, st>>>(sm, pm, rm, lay, g_first, n_gens)
#if CAO_GEN_ALGO == 2
    if (lay.wide && roww == 4 && threads <= 256) {
        k_gen<2, 4, 256, true><<<grid, threads, smem, st>>>(sm, pm, rm, lay, g_first, n_gens);
        CAO_LAUNCHED("k_gen");
        return CAO_OK;
    }
#endif
    if (roww == 4) { if (threads <= 256) LAUNCH(4, 256); else LAUNCH(4, 1024); }
    else           { if (threads <= 256) LAUNCH(8, 256); else LAUNCH(8, 1024); }
#undef LAUNCH
    CAO_LAUNCHED("k_gen");
    return CAO_OK;
}
