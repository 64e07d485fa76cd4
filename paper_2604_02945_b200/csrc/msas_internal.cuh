// msas_internal.cuh — device-side tables and small device helpers shared by the libmsas kernels.
// (CUDA path only.  The CPU oracle under oracle/ shares nothing with this tree.)
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace msas {

constexpr int kMaxL = 128;            // MAS_MAX_QUERY_TOKENS
constexpr int kTileRows = 128;        // rows per score tile (never straddles a segment)

// Device image of one segment (SPEC "Data model").
struct DevSeg {
  int64_t row0;
  int64_t kept_off_static;   // top-k mode: exclusive prefix of keep_k (host-known)
  int32_t n_rows;            // T*P
  int32_t n_patches;         // P
  int32_t n_frames;          // T
  int32_t request;
  int32_t q0;                // first query row of the request
  int32_t L;                 // query tokens of the request
  int32_t keep_k;
  int32_t tile0;             // index of the segment's first generic tile (DevTile table)
};

// One score tile: up to kTileRows consecutive rows of one segment.
struct DevTile {
  int32_t row_start;         // global row id
  int32_t n_rows;            // 1..kTileRows
  int32_t seg;
  int32_t pad_;
};

struct DevParams {
  float lambda_spatial, lambda_temp, tau_s, kappa;
  float spatial_gain, spatial_bias, rel_gain, rel_bias;
  float cut;
  int32_t select_mode;
};

// ---------------------------------------------------------------- small device helpers
__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
__device__ __forceinline__ float quad_sum(float v) {
  v += __shfl_xor_sync(0xffffffffu, v, 1);
  v += __shfl_xor_sync(0xffffffffu, v, 2);
  return v;
}
__device__ __forceinline__ float quad_max(float v) {
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 1));
  v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, 2));
  return v;
}

// streaming 16-byte load (read-only path, do not allocate in L1)
__device__ __forceinline__ uint4 ld_nc16(const void* p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "l"(p));
  return r;
}
__device__ __forceinline__ void st_na16(void* p, const uint4& v) {
  asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// packed bf16x2 -> two fp32 (exact)
__device__ __forceinline__ float bf_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf_hi(uint32_t u) { return __uint_as_float(u & 0xffff0000u); }

// fp32 pair -> packed bf16x2 (round to nearest even), low half = a
__device__ __forceinline__ uint32_t pack_bf16x2(float a, float b) {
  uint32_t r;
  asm("cvt.rn.bf16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(b), "f"(a));
  return r;
}

// order-preserving fp32 -> u32 key (ascending)
__device__ __forceinline__ uint32_t float_key(float f) {
  uint32_t u = __float_as_uint(f + 0.0f);   // -0 -> +0 so that equal values share one key
  return (u & 0x80000000u) ? ~u : (u | 0x80000000u);
}

// programmatic dependent launch (no-ops when the kernel was launched without the attribute): wait for the preceding kernel's results / let the next kernel's CTAs be scheduled
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// host: launch `kernel` on `st`, optionally with programmatic stream serialization behind the previous kernel in the stream
template <class... KArgs, class... Args>
inline cudaError_t launch_k(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, bool pdl, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
// same, with thread-block clusters of `cluster` CTAs along x (grid.x must be a multiple of it)
template <class... KArgs, class... Args>
inline cudaError_t launch_kc(void (*kernel)(KArgs...), dim3 grid, dim3 block, int cluster, cudaStream_t st, bool pdl, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = (unsigned)cluster; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = attr; cfg.numAttrs = pdl ? 2 : 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

__device__ __forceinline__ float sigmoidf_acc(float u) { return 1.0f / (1.0f + expf(-u)); }

}  // namespace msas
