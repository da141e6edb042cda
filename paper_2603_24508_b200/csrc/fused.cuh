// fused.cuh -- single-pass push+arrange.
#pragma once
#include "pic_device.cuh"

namespace pic {

struct FusedScratch {
    unsigned long long *block_state = nullptr; // look-back words, one per block (+ ticket)
    int *cell_bound = nullptr;                 // first owned cell of each block (+1 sentinel)
    int nblocks_cap = 0;
};

static inline int fused_alloc(FusedScratch &f, int nc, long long capacity)
{
    (void)f; (void)nc; (void)capacity;
    return 0;
}

} // namespace pic
