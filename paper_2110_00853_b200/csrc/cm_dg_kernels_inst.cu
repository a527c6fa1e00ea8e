// cm_dg_kernels_inst.cu -- instantiates the hot kernels for ONE polynomial order (compile with -DCM_NQ=<N+1>),
// so that the orders build in parallel.  Exposes cm_launch_gradient_nq<NQ> / cm_launch_tendency_nq<NQ>.
#include "cm_dg_kernels2.cuh"
#include "cm_dg_kernels3.cuh"
#include "cm_dg_kernels4.cuh"
#include "cm_dg_kernels5.cuh"

#ifndef CM_NQ
#error "compile with -DCM_NQ=<N+1>"
#endif

#define CM_CAT2(a, b) a##b
#define CM_CAT(a, b) CM_CAT2(a, b)
#define CM_HAS_V3 (CM_NQ <= CM_V3_MAXNQ)
#define CM_HAS_V4 (CM_NQ <= CM_V4_MAXNQ)

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

#if CM_HAS_V3
// one wave of resident CTAs: occupancy (CTAs per SM) x SM count, capped by the number of work units
template <typename K>
cudaError_t wave_size(K kernel, int threads, size_t smem, int& ctas) {
  int dev = 0, sms = 0, per_sm = 0;
  cudaError_t err = cudaGetDevice(&dev);
  if (err == cudaSuccess) err = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (err == cudaSuccess) err = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem);
  if (err == cudaSuccess && per_sm < 1) err = cudaErrorLaunchOutOfResources;
  ctas = sms * per_sm;
  return err;
}

template <int Nq, bool MOIST>
cudaError_t launch_grad3(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg3<Nq, MOIST>;
  static bool configured = false;
  static int wave = 0;
  if (!configured) {
    cudaError_t err = configure(cm3_gradient_kernel<Nq, MOIST>, C::GRAD_SMEM, configured);
    if (err == cudaSuccess) err = wave_size(cm3_gradient_kernel<Nq, MOIST>, C::THREADS, C::GRAD_SMEM, wave);
    if (err != cudaSuccess) { configured = false; return err; }
  }
  const int blocks = kp.n_units < wave ? kp.n_units : wave;
  cm3_gradient_kernel<Nq, MOIST><<<blocks, C::THREADS, C::GRAD_SMEM, st>>>(kp);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, bool SGS>
cudaError_t launch_tend3(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg3<Nq, MOIST>;
  static bool configured = false;
  static int wave = 0;
  if (!configured) {
    cudaError_t err = configure(cm3_tendency_kernel<Nq, MOIST, SGS>, C::TEND_SMEM, configured);
    if (err == cudaSuccess) err = wave_size(cm3_tendency_kernel<Nq, MOIST, SGS>, C::THREADS, C::TEND_SMEM, wave);
    if (err != cudaSuccess) { configured = false; return err; }
  }
  const int blocks = kp.n_units < wave ? kp.n_units : wave;
  cm3_tendency_kernel<Nq, MOIST, SGS><<<blocks, C::THREADS, C::TEND_SMEM, st>>>(kp);
  return cudaGetLastError();
}
#endif

template <int Nq, bool MOIST>
cudaError_t launch_grad5(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg5<Nq, MOIST>;
  static bool configured = false;
  cudaError_t err = configure(cm5_gradient_kernel<Nq, MOIST>, C::GRAD_SMEM, configured);
  if (err != cudaSuccess) return err;
  cm5_gradient_kernel<Nq, MOIST><<<kp.Ne, C::THREADS, C::GRAD_SMEM, st>>>(kp);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, bool SGS>
cudaError_t launch_tend5(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg5<Nq, MOIST>;
  static bool configured = false;
  cudaError_t err = configure(cm5_tendency_kernel<Nq, MOIST, SGS>, C::TEND_SMEM, configured);
  if (err != cudaSuccess) return err;
  cm5_tendency_kernel<Nq, MOIST, SGS><<<kp.Ne, C::THREADS, C::TEND_SMEM, st>>>(kp);
  return cudaGetLastError();
}

#if CM_HAS_V4
template <int Nq, bool MOIST>
cudaError_t launch_grad4(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg4<Nq, MOIST>;
  static bool configured = false;
  cudaError_t err = configure(cm4_gradient_kernel<Nq, MOIST>, C::GRAD_SMEM, configured);
  if (err != cudaSuccess) return err;
  const int per_cta = C::WG * kp.epw;
  cm4_gradient_kernel<Nq, MOIST><<<(kp.Ne + per_cta - 1) / per_cta, 32 * C::WG, C::GRAD_SMEM, st>>>(kp);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, bool SGS>
cudaError_t launch_tend4(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg4<Nq, MOIST>;
  static bool configured = false;
  cudaError_t err = configure(cm4_tendency_kernel<Nq, MOIST, SGS>, C::TEND_SMEM, configured);
  if (err != cudaSuccess) return err;
  const int per_cta = C::WT * kp.epw;
  cm4_tendency_kernel<Nq, MOIST, SGS><<<(kp.Ne + per_cta - 1) / per_cta, 32 * C::WT, C::TEND_SMEM, st>>>(kp);
  return cudaGetLastError();
}
#endif

}  // namespace

cudaError_t CM_CAT(cm_launch_gradient_nq, CM_NQ)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st) {
  if (variant == 5 && !general) return moist ? launch_grad5<CM_NQ, true>(kp, st) : launch_grad5<CM_NQ, false>(kp, st);
#if CM_HAS_V4
  if (variant == 4 && !general) return moist ? launch_grad4<CM_NQ, true>(kp, st) : launch_grad4<CM_NQ, false>(kp, st);
#endif
#if CM_HAS_V3
  if (variant == 3 && !general) return moist ? launch_grad3<CM_NQ, true>(kp, st) : launch_grad3<CM_NQ, false>(kp, st);
#endif
  if (moist) return general ? launch_grad2<CM_NQ, true, 1>(kp, st) : launch_grad2<CM_NQ, true, 0>(kp, st);
  return general ? launch_grad2<CM_NQ, false, 1>(kp, st) : launch_grad2<CM_NQ, false, 0>(kp, st);
}

cudaError_t CM_CAT(cm_launch_tendency_nq, CM_NQ)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st) {
  if (variant == 5 && !general) {
    if (kp.sgs) return moist ? launch_tend5<CM_NQ, true, true>(kp, st) : launch_tend5<CM_NQ, false, true>(kp, st);
    return moist ? launch_tend5<CM_NQ, true, false>(kp, st) : launch_tend5<CM_NQ, false, false>(kp, st);
  }
#if CM_HAS_V4
  if (variant == 4 && !general) {
    if (kp.sgs) return moist ? launch_tend4<CM_NQ, true, true>(kp, st) : launch_tend4<CM_NQ, false, true>(kp, st);
    return moist ? launch_tend4<CM_NQ, true, false>(kp, st) : launch_tend4<CM_NQ, false, false>(kp, st);
  }
#endif
#if CM_HAS_V3
  if (variant == 3 && !general) {
    if (kp.sgs) return moist ? launch_tend3<CM_NQ, true, true>(kp, st) : launch_tend3<CM_NQ, false, true>(kp, st);
    return moist ? launch_tend3<CM_NQ, true, false>(kp, st) : launch_tend3<CM_NQ, false, false>(kp, st);
  }
#endif
  if (moist) return general ? launch_tend2<CM_NQ, true, 1>(kp, st) : launch_tend2<CM_NQ, true, 0>(kp, st);
  return general ? launch_tend2<CM_NQ, false, 1>(kp, st) : launch_tend2<CM_NQ, false, 0>(kp, st);
}
