// round2.cu -- the translation unit of the device-launched second round (round2.cuh).
//
// Device-side launches need relocatable device code (-rdc=true), and relocatable device code costs the frame's main
// kernels dearly (measured on the B200: preprocess 0.077 -> 0.118 ms, blend 0.146 -> 0.153 ms when the whole library
// was built that way). So only this file is: it holds its OWN copies of the kernels the second round launches, in
// namespace pvg_r2 (the macro below renames the namespace of every header it includes), the gate kernel that launches
// them, and one host entry point, pvg_r2_gate, that pvg_api.cu calls through a plain C signature. The structures that
// cross the boundary (FrameParams, R2Chain, BlendLazy) come from the same headers on both sides: same layout.
#define pvg pvg_r2
#define PVG_NO_GRIDDEP 1   // launched from the device, never as programmatic dependents: no griddepcontrol
#include "round2.cuh"

#include <atomic>

namespace {
std::atomic<unsigned> g_ready{0};   // devices whose kernels have their shared-memory limit raised

template <class K>
cudaError_t ensure_smem(K kern, size_t bytes) {
  return bytes > 48 * 1024 ? cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes) : cudaSuccess;
}

template <int BITS>
cudaError_t ensure_emit() { return ensure_smem(pvg::bin_emit_kernel<BITS, false>, sizeof(pvg::BinEmitSmem<BITS>)); }

cudaError_t ensure_all() {
  using namespace pvg;
  cudaError_t e = ensure_smem(depth_pass_kernel<PVG_DS_THREADS, PVG_DS_ITEMS, DS_BITS, PVG_DS_MINB, false, true>,
                              sizeof(OnesweepSmem<PVG_DS_THREADS, PVG_DS_ITEMS, DS_BITS>));
  if (e == cudaSuccess)
    e = ensure_smem(depth_pass_kernel<PVG_DS_THREADS, PVG_DS_ITEMS, DS_TOP_BITS, PVG_DS_MINB, false, true>,
                    sizeof(OnesweepSmem<PVG_DS_THREADS, PVG_DS_ITEMS, DS_TOP_BITS>));
  if (e == cudaSuccess) e = ensure_emit<1>();
  if (e == cudaSuccess) e = ensure_emit<2>();
  if (e == cudaSuccess) e = ensure_emit<3>();
  if (e == cudaSuccess) e = ensure_emit<4>();
  if (e == cudaSuccess) e = ensure_emit<5>();
  if (e == cudaSuccess) e = ensure_emit<6>();
  if (e == cudaSuccess) e = ensure_emit<7>();
  if (e == cudaSuccess) e = ensure_emit<8>();
  return e;
}
}  // namespace

// Enqueues the gate on `stream` (after the first blend phase). params / chain / lazy: FrameParams, R2Chain, BlendLazy
// of the frame, by address (copied into the launch). which = COUNT * 3 + MODE of the frame's blend kernels.
// pdl: launch as a programmatic dependent of the kernel enqueued just before (the first blend phase). Returns a cudaError_t.
extern "C" int pvg_r2_gate(int device, void* stream, const void* params, const void* chain, const void* lazy, int which,
                           const void* ranges, const void* vals, const void* record, float* out_rgb, float* out_depth,
                           float* out_alpha, unsigned long long* counters, const float* featw, int pdl) {
  const unsigned bit = 1u << (device & 31);
  if (!(g_ready.load(std::memory_order_acquire) & bit)) {
    cudaError_t e = ensure_all();
    if (e != cudaSuccess) return (int)e;
    g_ready.fetch_or(bit, std::memory_order_release);
  }
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(1); cfg.blockDim = dim3(1); cfg.dynamicSmemBytes = 0; cfg.stream = (cudaStream_t)stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = pdl ? 1 : 0;   // only when the operation before it on the stream is the blend kernel
  cudaError_t e = cudaLaunchKernelEx(&cfg, pvg::r2_gate_kernel, *static_cast<const pvg::FrameParams*>(params),
                                     *static_cast<const pvg::R2Chain*>(chain), which, static_cast<const uint2*>(ranges),
                                     static_cast<const uint32_t*>(vals), static_cast<const float4*>(record), out_rgb, out_depth,
                                     out_alpha, counters, featw, *static_cast<const pvg::BlendLazy*>(lazy));
  return (int)(e != cudaSuccess ? e : cudaGetLastError());
}
