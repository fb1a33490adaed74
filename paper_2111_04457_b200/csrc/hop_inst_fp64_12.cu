// hop_inst_fp64_12.cu — every hop-kernel variant for fp64 storage, 12-real links (see hop_kernels.cuh).
#include "hop_kernels.cuh"

template bq_status launch_hop<BQ_FP64, BQ_RECON12>(bq_lattice*, void*, const void*, const void*, double, int, const void*, const void*, int,
                                                 const HopRed*, cudaStream_t, const HopMulti*, bool);
