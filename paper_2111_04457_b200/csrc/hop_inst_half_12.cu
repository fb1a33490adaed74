// hop_inst_half_12.cu — every hop-kernel variant for half storage, 12-real links (see hop_kernels.cuh).
#include "hop_kernels.cuh"

template bq_status launch_hop<BQ_HALF, BQ_RECON12>(bq_lattice*, void*, const void*, const void*, double, int, const void*, const void*, int,
                                                 const HopRed*, cudaStream_t, const HopMulti*, bool);
