// cm_dg_kernels_inst.cu -- instantiates the hot kernels for ONE polynomial order (compile with -DCM_NQ=<N+1>),
// so that the orders build in parallel.  Exposes cm_launch_gradient_nq<NQ> / cm_launch_tendency_nq<NQ>.
#include <atomic>
#include "cm_dg_kernels2.cuh"
#include "cm_dg_kernels7.cuh"
#include "cm_dg_kernels10.cuh"
#include "cm_dg_kernels11.cuh"

#ifndef CM_NQ
#error "compile with -DCM_NQ=<N+1>"
#endif

#define CM_CAT2(a, b) a##b
#define CM_CAT(a, b) CM_CAT2(a, b)

namespace {

template <int Nq, bool MOIST, bool RICH>
constexpr size_t grad2_smem() {
  using C = CmCfg2<Nq>;
  constexpr int NS = (MOIST ? 5 : 4) + (RICH ? 1 : 0);
  return sizeof(double) * (size_t)(4 * C::EPB * NS * C::NP + C::EPB * 6 * C::NF * NS);
}
template <int Nq, bool MOIST>
constexpr size_t tend2_smem() {
  using C = CmCfg2<Nq>;
  constexpr int NV = MOIST ? 6 : 5;
  return sizeof(double) * (size_t)(4 * C::EPB * NV * C::NP + C::EPB * C::NP + C::EPB * 6 * C::NF * NV);
}

// Per-kernel launch state, kept PER DEVICE: cudaFuncSetAttribute and the occupancy query act on the current device only.
// Concurrent first launches from several host threads at worst repeat the (idempotent) configuration.
constexpr int CM_MAX_DEVICES = 64;
struct LaunchState { std::atomic<bool> configured[CM_MAX_DEVICES]; std::atomic<int> wave[CM_MAX_DEVICES]; };

inline int current_device() { int dev = 0; cudaGetDevice(&dev); return (dev >= 0 && dev < CM_MAX_DEVICES) ? dev : 0; }

// one wave of resident CTAs = the L2 prefetch distance of the flat kernels (CmKP::ahead < 0)
template <typename K>
int wave_size(K kernel, int threads, size_t smem) {
  int dev = 0, sms = 0, per_sm = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
      cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, threads, smem) != cudaSuccess) return 0;
  return sms * per_sm;
}

// sets the shared-memory attributes of `kernel` on the current device once; returns the device's wave size in *wave
template <typename K>
cudaError_t configure(K kernel, size_t smem, LaunchState& ls, int threads = 0, int* wave = nullptr) {
  const int dev = current_device();
  if (!ls.configured[dev].load(std::memory_order_acquire)) {
    cudaError_t err = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (err == cudaSuccess) err = cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (err != cudaSuccess) return err;
    if (threads > 0) ls.wave[dev].store(wave_size(kernel, threads, smem), std::memory_order_relaxed);
    ls.configured[dev].store(true, std::memory_order_release);
  }
  if (wave) *wave = ls.wave[dev].load(std::memory_order_relaxed);
  return cudaSuccess;
}

template <int Nq, bool MOIST, int GEOM, bool RICH, bool SAT = false>
cudaError_t launch_grad2r(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg2<Nq>;
  static LaunchState ls;
  constexpr size_t smem = grad2_smem<Nq, MOIST, RICH>();
  int wave = 0;
  cudaError_t err = configure(cm2_gradient_kernel<Nq, MOIST, GEOM, RICH, SAT>, smem, ls, C::THREADS, &wave);
  if (err != cudaSuccess) return err;
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  CmKP k2 = kp;
  if (k2.ahead < 0) k2.ahead = wave * C::EPB;   // L2 prefetch distance in elements: one wave of resident CTAs
  cm2_gradient_kernel<Nq, MOIST, GEOM, RICH, SAT><<<blocks, C::THREADS, smem, st>>>(k2);
  return cudaGetLastError();
}
template <int Nq, bool MOIST, int GEOM>
cudaError_t launch_grad2(const CmKP& kp, cudaStream_t st) {
  // the Richardson factor (eq. 40) needs theta_v as a further gradient variable; the raw-gradient mode does not
  if constexpr (MOIST) {   // saturation-adjusted equation of state (eq. 15): its own instantiations
    if (kp.satadj) return (kp.richardson && kp.mode == 0) ? launch_grad2r<Nq, MOIST, GEOM, true, true>(kp, st) : launch_grad2r<Nq, MOIST, GEOM, false, true>(kp, st);
  }
  if (kp.richardson && kp.mode == 0) return launch_grad2r<Nq, MOIST, GEOM, true>(kp, st);
  return launch_grad2r<Nq, MOIST, GEOM, false>(kp, st);
}

template <int Nq, bool MOIST, int GEOM, bool SAT = false>
cudaError_t launch_tend2(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg2<Nq>;
  if constexpr (MOIST && !SAT) { if (kp.satadj) return launch_tend2<Nq, MOIST, GEOM, true>(kp, st); }
  static LaunchState ls;
  constexpr size_t smem = tend2_smem<Nq, MOIST>();
  int wave = 0;
  cudaError_t err = configure(cm2_tendency_kernel<Nq, MOIST, GEOM, SAT>, smem, ls, C::THREADS, &wave);
  if (err != cudaSuccess) return err;
  const int blocks = (kp.Ne + C::EPB - 1) / C::EPB;
  CmKP k2 = kp;
  if (k2.ahead < 0) k2.ahead = wave * C::EPB;   // L2 prefetch distance in elements: one wave of resident CTAs
  cm2_tendency_kernel<Nq, MOIST, GEOM, SAT><<<blocks, C::THREADS, smem, st>>>(k2);
  return cudaGetLastError();
}


template <int Nq, bool MOIST, bool RAW, bool GEM = false, bool RICH = false>
cudaError_t launch_grad7(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg7<Nq, MOIST>;
  static LaunchState ls;
  const dim3 grid(kp.gPY * kp.gL, kp.gEz, kp.gNXC * kp.gNYP);
  int wave = 0;
  CmKP k2 = kp;
  if constexpr (CmCfg9<Nq, MOIST>::OK) {
    // every line task has its own thread: register-staged traces (cm9_gradient_kernel)
    constexpr size_t smem = CmCfg9<Nq, MOIST>::GRAD_SMEM;
    cudaError_t err = configure(cm9_gradient_kernel<Nq, MOIST, RAW, GEM, RICH>, smem, ls, C::THREADS, &wave);
    if (err != cudaSuccess) return err;
    if (k2.ahead < 0) k2.ahead = wave;
    cm9_gradient_kernel<Nq, MOIST, RAW, GEM, RICH><<<grid, C::THREADS, smem, st>>>(k2);
  } else {
    cudaError_t err = configure(cm7_gradient_kernel<Nq, MOIST, RAW, GEM>, C::GRAD_SMEM, ls, C::THREADS, &wave);
    if (err != cudaSuccess) return err;
    if (k2.ahead < 0) k2.ahead = wave;
    cm7_gradient_kernel<Nq, MOIST, RAW, GEM><<<grid, C::THREADS, C::GRAD_SMEM, st>>>(k2);
  }
  return cudaGetLastError();
}

template <int Nq, bool MOIST, bool SGS, int MODE>
cudaError_t launch_tend7(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg7<Nq, MOIST>;
  static LaunchState ls;
  int wave = 0;
  cudaError_t err = configure(cm7_tendency_kernel<Nq, MOIST, SGS, MODE>, C::TEND_SMEM, ls, C::THREADS, &wave);
  if (err != cudaSuccess) return err;
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
    static LaunchState ls;
    cudaError_t err = configure(cm10_tendency_kernel<Nq, MOIST, SGS, MODE>, R::SMEM, ls);
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

// CTA-per-element tendency kernel of stored-metric meshes (cm_dg_kernels11.cuh): grid = the tiled element order
template <int Nq, bool MOIST, bool SGS, int MODE, bool TERR>
cudaError_t launch_tend11(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg7<Nq, MOIST>;
  using R = CmCfg11<Nq, MOIST, SGS, MODE, TERR>;
  static LaunchState ls;
  int wave = 0;
  cudaError_t err = configure(cm11_tendency_kernel<Nq, MOIST, SGS, MODE, TERR>, R::SMEM, ls, C::THREADS, &wave);
  if (err != cudaSuccess) return err;
  CmKP k2 = kp;
  if (k2.ahead < 0) k2.ahead = wave;
  cm11_tendency_kernel<Nq, MOIST, SGS, MODE, TERR><<<dim3(kp.gPY * kp.gL, kp.gEz, kp.gNXC * kp.gNYP), C::THREADS, R::SMEM, st>>>(k2);
  return cudaGetLastError();
}

template <int Nq, bool MOIST, bool RAW, bool RICH>
cudaError_t launch_grad11(const CmKP& kp, cudaStream_t st) {
  using C = CmCfg7<Nq, MOIST>;
  using R = CmCfg11G<Nq, MOIST, RICH>;
  static LaunchState ls;
  int wave = 0;
  cudaError_t err = configure(cm11_gradient_kernel<Nq, MOIST, RAW, RICH>, R::SMEM, ls, C::THREADS, &wave);
  if (err != cudaSuccess) return err;
  CmKP k2 = kp;
  if (k2.ahead < 0) k2.ahead = wave;
  cm11_gradient_kernel<Nq, MOIST, RAW, RICH><<<dim3(kp.gPY * kp.gL, kp.gEz, kp.gNXC * kp.gNYP), C::THREADS, R::SMEM, st>>>(k2);
  return cudaGetLastError();
}

template <int Nq, bool MOIST>
cudaError_t launch_grad11m(const CmKP& kp, cudaStream_t st) {
  if (kp.mode == 1) return launch_grad11<Nq, MOIST, true, false>(kp, st);
  return kp.richardson ? launch_grad11<Nq, MOIST, false, true>(kp, st) : launch_grad11<Nq, MOIST, false, false>(kp, st);
}

template <int Nq, bool MOIST, bool SGS, bool TERR>
cudaError_t launch_tend11t(const CmKP& kp, cudaStream_t st) {
  if (kp.mode == 0) return launch_tend11<Nq, MOIST, SGS, 0, TERR>(kp, st);
  return (kp.rka != 0.0) ? launch_tend11<Nq, MOIST, SGS, 1, TERR>(kp, st) : launch_tend11<Nq, MOIST, SGS, 2, TERR>(kp, st);
}

template <int Nq, bool MOIST, bool SGS>
cudaError_t launch_tend11m(const CmKP& kp, cudaStream_t st) {   // terrain-following meshes: three metric tiles instead of nine
  return kp.terrain ? launch_tend11t<Nq, MOIST, SGS, true>(kp, st) : launch_tend11t<Nq, MOIST, SGS, false>(kp, st);
}

}  // namespace

cudaError_t CM_CAT(cm_launch_gradient_nq, CM_NQ)(const CmKP& kp, int moist, int general, int variant, cudaStream_t st) {
  if ((variant == 7 || variant == 10) && !general) {
    if (kp.mode == 1) return moist ? launch_grad7<CM_NQ, true, true>(kp, st) : launch_grad7<CM_NQ, false, true>(kp, st);
    // (cm_dg_setup routes richardson = 1 to the thread-per-node kernels at the orders without a cm9 kernel)
    if (variant == 10 && CmCfg10<CM_NQ, true, 1>::OK) {   // the row-sweep tendency kernel reads G element-major
      if (kp.richardson) return moist ? launch_grad7<CM_NQ, true, false, true, true>(kp, st) : launch_grad7<CM_NQ, false, false, true, true>(kp, st);
      return moist ? launch_grad7<CM_NQ, true, false, true>(kp, st) : launch_grad7<CM_NQ, false, false, true>(kp, st);
    }
    if (kp.richardson) return moist ? launch_grad7<CM_NQ, true, false, false, true>(kp, st) : launch_grad7<CM_NQ, false, false, false, true>(kp, st);
    return moist ? launch_grad7<CM_NQ, true, false>(kp, st) : launch_grad7<CM_NQ, false, false>(kp, st);
  }
  if constexpr (CmCfg11G<CM_NQ, true, true>::OK) {
    if (variant == 11 && general) return moist ? launch_grad11m<CM_NQ, true>(kp, st) : launch_grad11m<CM_NQ, false>(kp, st);
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
  if constexpr (CmCfg11<CM_NQ, true, true, 1, false>::OK) {   // one predicate per order
    if (variant == 11 && general) {
      if (kp.sgs) return moist ? launch_tend11m<CM_NQ, true, true>(kp, st) : launch_tend11m<CM_NQ, false, true>(kp, st);
      return moist ? launch_tend11m<CM_NQ, true, false>(kp, st) : launch_tend11m<CM_NQ, false, false>(kp, st);
    }
  }
  if (moist) return general ? launch_tend2<CM_NQ, true, 1>(kp, st) : launch_tend2<CM_NQ, true, 0>(kp, st);
  return general ? launch_tend2<CM_NQ, false, 1>(kp, st) : launch_tend2<CM_NQ, false, 0>(kp, st);
}
