// cm_dg_kernels_inst.cu -- instantiates the hot kernels for ONE polynomial order (compile with -DCM_NQ=<N+1>),
// so that the orders build in parallel.  Exposes cm_launch_gradient_nq<NQ> / cm_launch_tendency_nq<NQ>.
#include "cm_dg_kernels2.cuh"
#include "cm_dg_kernels7.cuh"
#include "cm_dg_kernels10.cuh"

#ifndef CM_NQ
#error "compile with -DCM_NQ=<N+1>"
#endif

#define CM_CAT2(a, b) a##b
#define CM_CAT(a, b) CM_CAT2(a, b)

namespace {

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

template <typename K>
cudaError_t configure(K kernel, size_t smem, bool& configured) {
  if (configured) return cudaSuccess;
  cudaError_t err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (err == cudaSuccess) err = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
  if (err == cudaSuccess) configured = true;
  return err;
}

template <int Nq, bool MOIST, int GEOM>
cudaError_t launch_grad2(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg2<Nq>;
  static bool configured = false;
  constexpr size_t smem = grad2_smem<Nq, MOIST>();
  cudaError_t err = configure(cm2_gradient_kernel<Nq, MOIST, GEOM>, smem, configured);
  if (err != cudaSuccess) return err;
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  cm2_gradient_kernel<Nq, MOIST, GEOM><<<blocks, C::THREADS, smem, st>>>(kp);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, int GEOM>
cudaError_t launch_tend2(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg2<Nq>;
  static bool configured = false;
  constexpr size_t smem = tend2_smem<Nq, MOIST>();
  cudaError_t err = configure(cm2_tendency_kernel<Nq, MOIST, GEOM>, smem, configured);
  if (err != cudaSuccess) return err;
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  cm2_tendency_kernel<Nq, MOIST, GEOM><<<blocks, C::THREADS, smem, st>>>(kp);
  return cudaGetLastError();
}


// one wave of resident CTAs = the L2 prefetch distance of the flat kernels (CmKP::ahead < 0)
template <typename K>
int wave_size(K kernel, int threads, size_t smem) {
  int dev = 0, sms = 0, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess) return 0;
  return sms * per_sm;
}

template <int Nq, bool MOIST, bool RAW, bool GEM = false>
cudaError_t launch_grad7(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg7<Nq, MOIST>;
  static bool configured = false;
  const dim3 grid(kp.gPY * kp.gL, kp.gEz, kp.gNXC * kp.gNYP);
  if constexpr (CmCfg9<Nq, MOIST>::OK) {
    // every line task has its own thread: register-staged traces (cm9_gradient_kernel)
    constexpr size_t smem = CmCfg9<Nq, MOIST>::GRAD_SMEM;
    static int wave = 0;
    const bool first = !configured;
    cudaError_t err = configure(cm9_gradient_kernel<Nq, MOIST, RAW, GEM>, smem, configured);
    if (err != cudaSuccess) return err;
    if (first) wave = wave_size(cm9_gradient_kernel<Nq, MOIST, RAW, GEM>, C::THREADS, smem);
    CmKP k2 = kp;
    if (k2.ahead < 0) k2.ahead = wave;
    cm9_gradient_kernel<Nq, MOIST, RAW, GEM><<<grid, C::THREADS, smem, st>>>(k2);
  } else {
    static int wave = 0;
    const bool first = !configured;
    cudaError_t err = configure(cm7_gradient_kernel<Nq, MOIST, RAW, GEM>, C::GRAD_SMEM, configured);
    if (err != cudaSuccess) return err;
    if (first) wave = wave_size(cm7_gradient_kernel<Nq, MOIST, RAW, GEM>, C::THREADS, C::GRAD_SMEM);
    CmKP k2 = kp;
    if (k2.ahead < 0) k2.ahead = wave;
    cm7_gradient_kernel<Nq, MOIST, RAW, GEM><<<grid, C::THREADS, C::GRAD_SMEM, st>>>(k2);
  }
  return cudaGetLastError();
}

template <int Nq, bool MOIST, bool SGS, int MODE>
cudaError_t launch_tend7(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg7<Nq, MOIST>;
  static bool configured = false;
  static int wave = 0;
  const bool first = !configured;
  cudaError_t err = configure(cm7_tendency_kernel<Nq, MOIST, SGS, MODE>, C::TEND_SMEM, configured);
  if (err != cudaSuccess) return err;
  if (first) wave = wave_size(cm7_tendency_kernel<Nq, MOIST, SGS, MODE>, C::THREADS, C::TEND_SMEM);
  CmKP k2 = kp;
  if (k2.ahead < 0) k2.ahead = wave;
  cm7_tendency_kernel<Nq, MOIST, SGS, MODE><<<dim3(kp.gPY * kp.gL, kp.gEz, kp.gNXC * kp.gNYP), C::THREADS, C::TEND_SMEM, st>>>(k2);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, bool SGS>
cudaError_t launch_tend7m(const CmKP& kp, cudaStream_t st) {
  if (kp.mode == 0) return launch_tend7<Nq, MOIST, SGS, 0>(kp, st);
  return (kp.rka != 0.0) ? launch_tend7<Nq, MOIST, SGS, 1>(kp, st) : launch_tend7<Nq, MOIST, SGS, 2>(kp, st);
}

// row-sweep tendency kernel (cm_dg_kernels10.cuh): grid = rows of gS x-adjacent elements
template <int Nq, bool MOIST, bool SGS, int MODE>
cudaError_t launch_tend10(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg7<Nq, MOIST>;
  using R = CmCfg10<Nq, MOIST, MODE>;
  if constexpr (CmCfg10<Nq, true, 1>::OK) {   // one predicate per order: G / residual layouts must agree across all launches of a ctx
    static bool configured = false;
    cudaError_t err = configure(cm10_tendency_kernel<Nq, MOIST, SGS, MODE>, R::SMEM, configured);
    if (err != cudaSuccess) return err;
    const dim3 grid(kp.gPY * (kp.gL / kp.gS), kp.gEz, kp.gNXC * kp.gNYP);
    cm10_tendency_kernel<Nq, MOIST, SGS, MODE><<<grid, C::THREADS + 32, R::SMEM, st>>>(kp);
    return cudaGetLastError();
  } else {
    return launch_tend7<Nq, MOIST, SGS, MODE>(kp, st);
  }
}

template <int Nq, bool MOIST, bool SGS>
cudaError_t launch_tend10m(const CmKP& kp, cudaStream_t st) {
  if (kp.mode == 0) return launch_tend10<Nq, MOIST, SGS, 0>(kp, st);
  return (kp.rka != 0.0) ? launch_tend10<Nq, MOIST, SGS, 1>(kp, st) : launch_tend10<Nq, MOIST, SGS, 2>(kp, st);
}

}  // namespace

cudaError_t CM_CAT(cm_launch_gradient_nq, CM_NQ)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st) {
  if ((variant == 7 || variant == 10) && !general) {
    if (kp.mode == 1) return moist ? launch_grad7<CM_NQ, true, true>(kp, st) : launch_grad7<CM_NQ, false, true>(kp, st);
    if (variant == 10 && CmCfg10<CM_NQ, true, 1>::OK)    // the row-sweep tendency kernel reads G element-major
      return moist ? launch_grad7<CM_NQ, true, false, true>(kp, st) : launch_grad7<CM_NQ, false, false, true>(kp, st);
    return moist ? launch_grad7<CM_NQ, true, false>(kp, st) : launch_grad7<CM_NQ, false, false>(kp, st);
  }
  if (moist) return general ? launch_grad2<CM_NQ, true, 1>(kp, st) : launch_grad2<CM_NQ, true, 0>(kp, st);
  return general ? launch_grad2<CM_NQ, false, 1>(kp, st) : launch_grad2<CM_NQ, false, 0>(kp, st);
}

cudaError_t CM_CAT(cm_launch_tendency_nq, CM_NQ)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st) {
  if (variant == 10 && !general) {
    if (kp.sgs) return moist ? launch_tend10m<CM_NQ, true, true>(kp, st) : launch_tend10m<CM_NQ, false, true>(kp, st);
    return moist ? launch_tend10m<CM_NQ, true, false>(kp, st) : launch_tend10m<CM_NQ, false, false>(kp, st);
  }
  if (variant == 7 && !general) {
    if (kp.sgs) return moist ? launch_tend7m<CM_NQ, true, true>(kp, st) : launch_tend7m<CM_NQ, false, true>(kp, st);
    return moist ? launch_tend7m<CM_NQ, true, false>(kp, st) : launch_tend7m<CM_NQ, false, false>(kp, st);
  }
  if (moist) return general ? launch_tend2<CM_NQ, true, 1>(kp, st) : launch_tend2<CM_NQ, true, 0>(kp, st);
  return general ? launch_tend2<CM_NQ, false, 1>(kp, st) : launch_tend2<CM_NQ, false, 0>(kp, st);
}
