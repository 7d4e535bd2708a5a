// pyr_inst.cu -- instantiates the kernels of one FFT size: compile with -DPYR_INST_N=<N>.
//   pyr_pick_set_<N>  : full-length table-mask kernels of length N
//   pyr_pick_half_<N> : half-band-split kernels for N_fft = N (transform length N/2), N >= 32
#include "pyr_kernels.cuh"

#ifndef PYR_INST_N
#error "compile with -DPYR_INST_N=<N_fft>"
#endif
#define PYR_CAT2(a, b) a##b
#define PYR_CAT(a, b) PYR_CAT2(a, b)

KernelSet PYR_CAT(pyr_pick_set_, PYR_INST_N)(int prune) { return pick_set<PYR_INST_N>(prune); }

HalfSet PYR_CAT(pyr_pick_half_, PYR_INST_N)(int prune) {
#if PYR_INST_N >= 32
    return pick_half_prune<PYR_INST_N / 2>(prune);
#else
    (void)prune;
    return HalfSet{};
#endif
}

#if PYR_INST_N == 2048
Gen2Set pyr_pick_gen2(int prune) { return prune == 4 ? make_gen2<4>() : prune == 2 ? make_gen2<2>() : make_gen2<1>(); }
#endif
