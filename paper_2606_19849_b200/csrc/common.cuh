// Shared host/device helpers of the vcs library (sm_100a only).  Not part of the public ABI.
#pragma once

#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda.h>
#include <stdint.h>
#include <stdio.h>
#include <stdarg.h>
#include <atomic>

#include "vcs.h"

namespace vcs {

// ---- error reporting ---------------------------------------------------------------------
void set_error(const char* fmt, ...);
#define VCS_FAIL(code, ...)            \
  do {                                 \
    ::vcs::set_error(__VA_ARGS__);     \
    return (code);                     \
  } while (0)

#define VCS_CUDA_OK(expr)                                                             \
  do {                                                                                \
    cudaError_t e__ = (expr);                                                         \
    if (e__ != cudaSuccess) VCS_FAIL(VCS_ECUDA, "%s: %s", #expr, cudaGetErrorString(e__)); \
  } while (0)

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
static inline size_t elem_bytes(int dtype) { return dtype == VCS_BF16 ? 2 : 4; }
static inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- host-side pool bookkeeping (lives in vcs_kv_pool::opaque_h) ---------------------------
struct PoolOpaque {
  uint32_t magic;
  int32_t has_tma;
  alignas(64) CUtensorMap tmap_k;   // 4-D (d, token, kv head, page), box (64, 64, 1, 1), SWIZZLE_128B
  alignas(64) CUtensorMap tmap_v;
  double inv_freq[64];              // theta^(-2m/d), m < d/2 (fp64: angle = pos * inv_freq is exact to 1 ulp)
  int8_t axis_of[64];               // 0/1/2 = t/h/w for pair m
};
constexpr uint32_t kPoolMagic = 0x56435331u;  // "VCS1"

// M-RoPE parameters passed to kernels by value.
struct RopeParams {
  double inv_freq[64];
  unsigned long long turn_frac[64];   // frac(inv_freq / 2 pi) as a Q0.64 fixed-point fraction of a turn
  int8_t axis_of[64];
  int half;  // d/2
};

unsigned long long turn_fraction_q64(double inv_freq);   // frac(inv_freq / 2 pi) in Q0.64 (RopeParams::turn_frac)
int validate_pool(const vcs_kv_pool* pool, bool need_opaque);
RopeParams rope_params(const vcs_kv_pool* pool);

// ---- per-device host state ------------------------------------------------------------------
// The library keeps no mutable state that changes results: what is remembered is per-DEVICE and
// idempotent (the SM count, and "cudaFuncSetAttribute already applied on this device"), in lock-free
// tables indexed by the CUDA device ordinal, so calls are re-entrant across threads, streams and devices.
constexpr int kMaxDevices = 64;
int device_sm_count();      // SMs of the CURRENT device; 0 if the query fails (callers return VCS_ECUDA)
struct PerDeviceOnce {
  std::atomic<unsigned long long> done{0ull};
  // runs fn() once per device (again after a failure); returns VCS_OK or VCS_ECUDA
  template <typename F>
  int run(F&& fn) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices) dev = 0;
    const unsigned long long bit = 1ull << dev;
    if (done.load(std::memory_order_acquire) & bit) return VCS_OK;
    const cudaError_t e = fn();
    if (e != cudaSuccess) VCS_FAIL(VCS_ECUDA, "cudaFuncSetAttribute: %s", cudaGetErrorString(e));
    done.fetch_or(bit, std::memory_order_release);
    return VCS_OK;
  }
};

// ---- device helpers -----------------------------------------------------------------------
#ifdef __CUDACC__

// Programmatic dependent launch: every vcs kernel is launched with the programmatic-stream-
// serialization attribute and begins with pdl_wait() (blocks until the preceding kernel of the
// stream has completed and its writes are visible) followed by pdl_launch_dependents() (lets the
// NEXT kernel's CTAs become resident and sit in their own pdl_wait()).  Nothing is read or
// written before the wait, so ordering is exactly that of a plain stream; what is hidden is the
// launch latency between the three dependent kernels of a chunk.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <typename... KArgs, typename... Args>
static inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st,
                                     Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

__device__ __forceinline__ uint4 ldg_nc_v4(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}
__device__ __forceinline__ void stg_v4(void* p, uint4 v) {
  asm volatile("st.global.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w)
               : "memory");
}
__device__ __forceinline__ float bf16_lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16_hi(uint32_t w) { return __uint_as_float(w & 0xFFFF0000u); }
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);
  return *reinterpret_cast<uint32_t*>(&v);
}

// sin/cos of pos * inv_freq with the angle formed and range-reduced in fp64 (positions reach
// 1e5; an fp32 angle of that size is only good to ~1e-3 rad); the reduced angle lies in
// [-pi, pi] where sincosf is accurate to ~1 ulp.
__device__ __forceinline__ void rope_sincos(int pos, double inv_freq, float* s, float* c) {
  const double two_pi = 6.283185307179586476925286766559;
  double a = (double)pos * inv_freq;
  a -= two_pi * rint(a * (1.0 / two_pi));
  sincosf((float)a, s, c);
}

// Two-level "last block" ticket.  Hundreds of same-address atomics from different SMs serialise
// in L2 (~27 cycles each), so blocks first count inside groups (>= 16 blocks, at most 63 groups)
// on counters 128 B apart; only the last block of each group touches the top-level counter.
// Call from ONE thread after a __syncthreads(); returns true in exactly one block per launch.
// The region is kTicketBytes long whatever the grid (so a workspace reused with other sizes
// never aliases it), must be zero on entry and is left zero.  Slot 0 = top level, 1 + g = group g.
constexpr int kTicketMaxGroups = 63;
constexpr size_t kTicketBytes = (size_t)(1 + kTicketMaxGroups) * 128;
__device__ __forceinline__ bool last_block_ticket(unsigned int* counters, int block, int nblocks) {
  const int gsz = max(16, (nblocks + kTicketMaxGroups - 1) / kTicketMaxGroups);
  const int grp = block / gsz;
  const int in_group = min(gsz, nblocks - grp * gsz);
  unsigned int* gc = counters + 32 * (1 + grp);
  __threadfence();
  if (atomicAdd(gc, 1u) != (unsigned)(in_group - 1)) return false;
  *gc = 0u;
  __threadfence();
  const int ngroups = (nblocks + gsz - 1) / gsz;
  if (atomicAdd(counters, 1u) != (unsigned)(ngroups - 1)) return false;
  *counters = 0u;
  __threadfence();
  return true;
}

// Fast form for results that are rounded to bf16 right after: the angle in TURNS is
// pos * frac(inv_freq / 2 pi) mod 1, formed exactly in Q0.64 fixed point by one 64-bit integer
// multiply (the wrap-around IS the range reduction; no fp64).  Its top 23 bits become the mantissa of a
// float in [1, 2) -- no integer-to-float conversion, which shares the quarter-rate XU pipe with MUFU --
// so the angle in [-pi, pi) is good to 2 pi 2^-24 = 3.7e-7 rad; MUFU sin / cos add ~5e-7 absolute.
__device__ __forceinline__ void rope_sincos_fast(int pos, unsigned long long turn_frac, float* s, float* c) {
  const unsigned long long t = (unsigned long long)(long long)pos * turn_frac;
  float f = __uint_as_float(0x3f800000u | (unsigned int)((t + (1ull << 40)) >> 41)) - 1.0f;   // fraction of a turn in [0, 1), rounded
  f = f >= 0.5f ? f - 1.0f : f;
  const float a = f * 6.283185307179586f;
  *s = __sinf(a);
  *c = __cosf(a);
}

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float warp_max(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
  return v;
}

#endif  // __CUDACC__

}  // namespace vcs
