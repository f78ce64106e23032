// Device helpers shared by the stage kernels (f4_stage.cu: Euler, f4_advect.cu: scalar advection): fast fp64
// reciprocal / rsqrt, mbarrier and bulk-copy (TMA engine) wrappers, the limited half slope.
#pragma once
#include <cstdint>

#include "../../include/f4.h"

namespace f4 {

// ---- fast fp64 reciprocal / rsqrt: MUFU seed (~2^-22) + one cubic step -> < 2 ulp (reading B1)
__device__ __forceinline__ double rcp_seed(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}
__device__ __forceinline__ double rsqrt_seed(double x) {
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  return r;
}
__device__ __forceinline__ double rcp_refine(double x, double r) {
  const double e = fma(-x, r, 1.0);
  const double e2 = fma(e, e, e);
  return fma(r, e2, r);
}
__device__ __forceinline__ double rsqrt_refine(double x, double y) {
  // y*y and y*e are formed beside the Newton terms: the dependent chain is DMUL, DFMA, DFMA/DMUL, DFMA
  const double e = fma(-x, y * y, 1.0);
  const double h = fma(0.375, e, 0.5);
  return fma(y * e, h, y);
}
__device__ __forceinline__ double rcp_fast(double x) { return rcp_refine(x, rcp_seed(x)); }
__device__ __forceinline__ double rsqrt_fast(double x) { return rsqrt_refine(x, rsqrt_seed(x)); }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// 1-D bulk async copy global -> shared (TMA engine; SASS UBLKCP), completion counted on the mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void group_sync(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// limited HALF slope 1/2*phi(a,b) for the reconstruction w +- 1/2 phi (reading A1)
template <bool FAST>
__device__ __forceinline__ double half_slope(double a, double b, int limiter) {
  double ab = a * b;
  if (FAST) {
    // van Leer: 1/2 * 2ab/(a+b) where ab > 0.  The sign test is taken on the high word of ab (an integer compare
    // instead of a DSETP on the fp64 pipe); it differs from ab > 0 only for 0 < ab < 2^-1042, where the slope is < 1e-150.
    // the select is taken on the MUFU seed (one 32-bit select: the seed's low word is zero): seed 0 -> rcp 0 -> slope 0
    const double x = a + b;
    double y = rcp_seed(x);
    y = __hiloint2double((__double2hiint(ab) > 0) ? __double2hiint(y) : 0, 0);
    const double e = fma(-x, y, 1.0);
    const double t = ab * y;             // beside the Newton terms, off the dependent chain
    const double e2 = fma(e, e, e);
    return fma(t, e2, t);
  }
  double r;
  if (limiter == F4_LIM_WENO3) {
    // third-order WENO towards the b side (reading A1b): candidates w + a/2, w + b/2, ideal weights
    // 1/3, 2/3, smoothness a^2, b^2, eps = 1e-6; no sign test (the weights do the limiting)
    const double ea = 1e-6 + a * a, eb = 1e-6 + b * b;
    const double a0 = (1.0 / 3.0) / (ea * ea), a1 = (2.0 / 3.0) / (eb * eb);
    return 0.5 * ((a0 * a + a1 * b) / (a0 + a1));
  }
  if (limiter == F4_LIM_VANLEER) {
    r = ab * rcp_fast(a + b);
  } else if (limiter == F4_LIM_KOREN) {
    // Koren (reading A1b): the kappa = 1/3 slope (a + 2b)/3 towards the b side, limited to [0,2a], [0,2b]
    double m = fmin(fmin(2.0 * fabs(a), (fabs(a) + 2.0 * fabs(b)) / 3.0), 2.0 * fabs(b));
    r = 0.5 * ((a > 0.0) ? m : -m);
  } else {
    double th = (limiter == F4_LIM_MC) ? 2.0 : 1.0;   // eq. (1)
    double m = fmin(fmin(fabs(th * a), fabs(th * b)), fabs(a + b) * 0.5);
    r = 0.5 * ((a > 0.0) ? m : -m);
  }
  return (ab > 0.0) ? r : 0.0;
}

}  // namespace f4
