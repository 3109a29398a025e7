// dia_eval_inst.cu -- one translation unit per kernel size: compiled once for every odd m with
// -DDIA_INST_M=<m> (paper_2104_13715_b200/build.py runs these compilations in parallel).  Each unit holds the
// five instantiations of the fused kernel for its m and its own copy of the constant block, and exports two
// accessors that dia_api.cu uses to launch the kernels and to address the constant symbol.
#include "dia_eval.cuh"
#include "dia_fit_cluster.cuh"
#include "dia_hess_tc.cuh"

#ifndef DIA_INST_M
#error "compile with -DDIA_INST_M=<odd kernel size>"
#endif

#define DIA_CAT2(a, b) a##b
#define DIA_CAT(a, b) DIA_CAT2(a, b)

namespace dia {

// variant: 0 = plain objective, 1 = generic (mask / flat / variance map), 2 = difference image,
//          3 = plain objective with the kernel pixels in the constant bank, 4 = kernel-kernel block of the Hessian,
//          5 = generic with the kernel pixels in the constant bank, 6 = whole fit of a small image in one cluster,
//          7 = kernel-kernel block of the Hessian on the tensor cores (null when its shared memory does not fit)
const void* DIA_CAT(eval_kernel_ptr_m, DIA_INST_M)(int variant) {
  switch (variant) {
    case 0: return (const void*)eval_kernel<DIA_INST_M, false, false, false>;
    case 1: return (const void*)eval_kernel<DIA_INST_M, true, false, false>;
    case 2: return (const void*)eval_kernel<DIA_INST_M, true, true, false>;
    case 3: return (const void*)eval_kernel<DIA_INST_M, false, false, true>;
    case 4: return (const void*)hess_block_kernel<DIA_INST_M>;
    case 5: return (const void*)eval_kernel<DIA_INST_M, true, false, true>;
    case 6: return (const void*)fit_cluster_kernel<DIA_INST_M>;
    case 7: return TcGeo<DIA_INST_M>::FITS ? (const void*)hess_tc_kernel<DIA_INST_M> : nullptr;
  }
  return nullptr;
}

// dynamic shared memory of fit_cluster_kernel and of hess_tc_kernel
size_t DIA_CAT(cluster_smem_m, DIA_INST_M)() { return ClusterGeo<DIA_INST_M>::SMEM; }
size_t DIA_CAT(hess_tc_smem_m, DIA_INST_M)() { return TcGeo<DIA_INST_M>::SMEM; }

// host shadow of this unit's constant block (what cudaMemcpyToSymbol / graph memcpy nodes take)
const void* DIA_CAT(const_symbol_m, DIA_INST_M)() { return (const void*)&c_blk; }

}  // namespace dia

#if defined(DIA_CLUSTER_PROFILE) && DIA_INST_M == 7
// profiling builds only (-DDIA_CLUSTER_PROFILE): the clock64 phase counters of fit_cluster_kernel<7>, CTA 0
extern "C" void dia_cluster_prof(long long* out, int reset) {
  if (reset) { long long z[16] = {}; cudaMemcpyToSymbol(dia::g_cl_prof, z, sizeof(z)); }
  else cudaMemcpyFromSymbol(out, dia::g_cl_prof, sizeof(long long) * 16);
}
#endif
