// common.cuh -- shared device/host definitions of the PVG CUDA path (sm_100a).
// Product code: shares nothing with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#define PVG_TILE 16
#define PVG_TILE_PIXELS 256

// contract constants: S6, S9
#define PVG_ALPHA_MIN 0.003921569f /* fp32(1/255) */
#define PVG_ALPHA_MAX 0.99f
#define PVG_T_STOP 1e-4f
#define PVG_DILATE 0.3f
#define PVG_DILATE_D 0.3 /* the same reading (S6) for the double-precision conic: 0.3 px^2, not fp32(0.3) */
#define PVG_ZNEAR_DEFAULT 0.2f

namespace pvg {

// Per-frame constants, passed by value as a __grid_constant__ kernel parameter.
struct FrameParams {
  // The position chain mu~(t) -> p_cam -> (mx, my) runs in double (preprocess.cuh): the time the state is evaluated
  // at (t - dts, exact) and the two constants of Eq. 6, computed by the host in double.
  double t1;          // t - dts
  double two_over_l;  // 2 / l: sin(2 pi dt / l) = sinpi(two_over_l * dt)   (0 for the linear model)
  double l_over_2pi;  // l / (2 pi)
  double inv_l_d;     // 1 / l (0 for the linear model), for the flow translation of Eq. 12
  double Rd[9], Td[3], fxd, fyd, cxd, cyd;   // the camera once more, as doubles (exact copies of the fp32 fields below)
  double limxd, limyd;                       // 1.3 * half-FoV tangents, unrounded
  float R[9];       // world->camera rotation, row-major
  float T[3];       // world->camera translation
  float campos[3];  // camera centre in world coordinates (-R^T T)
  float fx, fy, cx, cy;
  float limx, limy;  // 1.3 * half-FoV tangents (Jacobian guard)
  float znear;
  float dts;          // Eq. 12 flow translation interval (0: the plain state H(t))
  float inv_l;        // 1 / l (0 for the linear model): rho = beta / l
  float rho_min, rho_max;  // staticness filter (only when `filter` is set)
  int filter;
  int cull;           // blend: drop list entries whose ellipse cannot reach the tile (bit-identical images)
  int target;         // 0: colour (SH) + depth; 1: dynamics -- colour := vbar in camera axes, 4th channel := clamp(rho, 0, 2)
  int linear;         // l == +INF: mu~ = mu + (t - tau) v
  int sh_degree;
  int width, height, tiles_x, tiles_y;
  int pack_rect;      // tiles_x, tiles_y <= 256: the depth key carries the tile rectangle in its upper half
  int band_y0, band_y1;  // tile rows [band_y0, band_y1) this render covers (the whole image: 0, tiles_y)
  float bg[3];
  const float* sky;   // cube map [6][res][res][3] or nullptr: rgb = C + (1 - O) f_sky(d)
  int sky_res;
  int lazy_slab;      // PVG_OPT_LAZY_SLAB (front-first depth order: preprocess sizes the front from it)
  uint32_t lazy_min_tiles;   // floor of the first slab in bin_emit tiles (lazy_emit_first)
};

// Lazy lists: bin_emit forms the block entries in tiles of PVG_EMIT_TILE (== BF_TILE, blockbin.cuh); its first launch
// takes the first 1 / lazy_slab of the tiles (at least one). One formula for the host and for preprocess's last CTA.
#define PVG_EMIT_TILE 4096
// min_tiles: a floor -- twice what the first LAZY_CHUNKS chunks of every block hold (FrameParams::lazy_min_tiles): the
// first round writes the lists as far as those chunks reach, and only chunks whose entries all exist count. At config 1
// (40 blocks, 78 tiles of entries) a sixteenth of the entries is half of that, and 800 of the 2400 tiles parked.
__host__ __device__ inline uint32_t lazy_emit_first(unsigned long long Mb, int lazy_slab, uint32_t min_tiles) {
  const uint32_t tiles = (uint32_t)((Mb + PVG_EMIT_TILE - 1) / PVG_EMIT_TILE);
  const uint32_t slab = lazy_slab > 0 ? (uint32_t)lazy_slab : 1u;
  uint32_t first = (tiles + slab - 1u) / slab;
  if (first < min_tiles) first = min_tiles;
  if (first < 1u) first = 1u;
  return tiles < first ? tiles : first;
}

__device__ __forceinline__ uint32_t lane_id() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%laneid;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%lanemask_lt;" : "=r"(r));
  return r;
}

// Programmatic dependent launch (sm_90+): a kernel launched with cudaLaunchAttributeProgrammaticStreamSerialization may
// start -- its CTAs become resident and run up to pdl_wait() -- while the kernel before it in the stream is still
// draining; pdl_wait() returns when that kernel has completed and its writes are visible. pdl_launch_dependents()
// lets the NEXT kernel of the stream do the same with respect to this one. Both are no-ops in a plain launch.
// Every kernel of a chain waits before its first global read (transitively, everything earlier has then completed).
// PVG_NO_GRIDDEP (round2.cu: the copies of the kernels that are launched from the device, never as programmatic
// dependents): both are empty.
#ifdef PVG_NO_GRIDDEP
__device__ __forceinline__ void pdl_wait() {}
__device__ __forceinline__ void pdl_launch_dependents() {}
#else
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif

// 64-bit status words of the decoupled look-back (flag in the top 2 bits, value
// below): one aligned 64-bit access carries flag and payload together, so relaxed
// gpu-scope accesses are sufficient.
__device__ __forceinline__ void st_relaxed_u64(uint64_t* p, uint64_t v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint64_t ld_relaxed_u64(const uint64_t* p) {
  uint64_t v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
constexpr uint64_t LB_FLAG_AGG = 1ull << 62;
constexpr uint64_t LB_FLAG_PREFIX = 2ull << 62;
constexpr uint64_t LB_FLAG_MASK = 3ull << 62;
constexpr uint64_t LB_VALUE_MASK = ~LB_FLAG_MASK;

// streaming (read-once) 128-bit load that does not allocate in L1
__device__ __forceinline__ float4 ldg_stream_f4(const float4* p) {
  float4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.f32 {%0,%1,%2,%3}, [%4];"
               : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
               : "l"(p));
  return v;
}

// corner updates of one rectangle [x0,x1] x [y0,y1] (inclusive) on the (TX+1) x (TY+1) grid
__device__ __forceinline__ void tilegrid_add_rect(int* __restrict__ grid, int stride, int x0, int y0, int x1, int y1) {
  atomicAdd(grid + y0 * stride + x0, 1);
  atomicAdd(grid + y0 * stride + x1 + 1, -1);
  atomicAdd(grid + (y1 + 1) * stride + x0, -1);
  atomicAdd(grid + (y1 + 1) * stride + x1 + 1, 1);
}

__host__ __device__ inline int tilegrid_stride(int tiles_x) { return (tiles_x + 1) | 1; }  // odd: conflict-free rows

}  // namespace pvg
