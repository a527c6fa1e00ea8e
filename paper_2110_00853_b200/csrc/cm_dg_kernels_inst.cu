// cm_dg_kernels_inst.cu -- instantiates the hot kernels for ONE polynomial order (compile with -DCM_NQ=<N+1>),
// so that the orders build in parallel.  Exposes cm_launch_gradient_nq<NQ> / cm_launch_tendency_nq<NQ>.
#include "cm_dg_kernels.cuh"
#include "cm_dg_kernels2.cuh"

#ifndef CM_NQ
#error "compile with -DCM_NQ=<N+1>"
#endif

#define CM_CAT2(a, b) a##b
#define CM_CAT(a, b) CM_CAT2(a, b)

namespace {

template <int Nq, bool MOIST>
constexpr size_t grad_smem() {
  using C = CmCfg<Nq>;
  constexpr int NS = MOIST ? 5 : 4;
  return sizeof(double) * (size_t)(Nq * Nq + C::EPB * NS * C::NP + C::EPB * 4 * C::NF * NS);
}
template <int Nq, bool MOIST>
constexpr size_t tend_smem() {
  using C = CmCfg<Nq>;
  constexpr int NV = MOIST ? 6 : 5;
  return sizeof(double) * (size_t)(Nq * Nq + 2 * C::EPB * NV * C::NP + C::EPB * C::NP + C::EPB * 4 * C::NF * NV);
}

template <int Nq, bool MOIST, int GEOM>
cudaError_t launch_grad(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg<Nq>;
  static bool configured = false;
  constexpr size_t smem = grad_smem<Nq, MOIST>();
  if (!configured) {
    cudaError_t err = cudaFuncSetAttribute(cm_gradient_kernel<Nq, MOIST, GEOM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    configured = true;
  }
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  cm_gradient_kernel<Nq, MOIST, GEOM><<<blocks, C::THREADS, smem, st>>>(kp);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, int GEOM>
cudaError_t launch_tend(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg<Nq>;
  static bool configured = false;
  constexpr size_t smem = tend_smem<Nq, MOIST>();
  if (!configured) {
    cudaError_t err = cudaFuncSetAttribute(cm_tendency_kernel<Nq, MOIST, GEOM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    configured = true;
  }
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  cm_tendency_kernel<Nq, MOIST, GEOM><<<blocks, C::THREADS, smem, st>>>(kp);
  return cudaGetLastError();
}

template <int Nq, bool MOIST>
constexpr size_t grad2_smem() {
  using C = CmCfg2<Nq>;
  constexpr int NS = MOIST ? 5 : 4;
  return sizeof(double) * (size_t)(4 * C::EPB * NS * C::NP + C::EPB * 6 * C::NF * NS);
}
template <int Nq, bool MOIST>
constexpr size_t tend2_smem() {
  using C = CmCfg2<Nq>;
  constexpr int NV = MOIST ? 6 : 5;
  return sizeof(double) * (size_t)(4 * C::EPB * NV * C::NP + C::EPB * C::NP + C::EPB * 6 * C::NF * NV);
}

template <int Nq, bool MOIST, int GEOM>
cudaError_t launch_grad2(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg2<Nq>;
  static bool configured = false;
  constexpr size_t smem = grad2_smem<Nq, MOIST>();
  if (!configured) {
    cudaError_t err = cudaFuncSetAttribute(cm2_gradient_kernel<Nq, MOIST, GEOM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    configured = true;
  }
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  cm2_gradient_kernel<Nq, MOIST, GEOM><<<blocks, C::THREADS, smem, st>>>(kp);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, int GEOM>
cudaError_t launch_tend2(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg2<Nq>;
  static bool configured = false;
  constexpr size_t smem = tend2_smem<Nq, MOIST>();
  if (!configured) {
    cudaError_t err = cudaFuncSetAttribute(cm2_tendency_kernel<Nq, MOIST, GEOM>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err != cudaSuccess) return err;
    configured = true;
  }
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  cm2_tendency_kernel<Nq, MOIST, GEOM><<<blocks, C::THREADS, smem, st>>>(kp);
  return cudaGetLastError();
}

}  // namespace

cudaError_t CM_CAT(cm_launch_gradient_nq, CM_NQ)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st) {
  if (variant == 1) {
    if (moist) return general ? launch_grad<CM_NQ, true, 1>(kp, st) : launch_grad<CM_NQ, true, 0>(kp, st);
    return general ? launch_grad<CM_NQ, false, 1>(kp, st) : launch_grad<CM_NQ, false, 0>(kp, st);
  }
  if (moist) return general ? launch_grad2<CM_NQ, true, 1>(kp, st) : launch_grad2<CM_NQ, true, 0>(kp, st);
  return general ? launch_grad2<CM_NQ, false, 1>(kp, st) : launch_grad2<CM_NQ, false, 0>(kp, st);
}

cudaError_t CM_CAT(cm_launch_tendency_nq, CM_NQ)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st) {
  if (variant == 1) {
    if (moist) return general ? launch_tend<CM_NQ, true, 1>(kp, st) : launch_tend<CM_NQ, true, 0>(kp, st);
    return general ? launch_tend<CM_NQ, false, 1>(kp, st) : launch_tend<CM_NQ, false, 0>(kp, st);
  }
  if (moist) return general ? launch_tend2<CM_NQ, true, 1>(kp, st) : launch_tend2<CM_NQ, true, 0>(kp, st);
  return general ? launch_tend2<CM_NQ, false, 1>(kp, st) : launch_tend2<CM_NQ, false, 0>(kp, st);
}
