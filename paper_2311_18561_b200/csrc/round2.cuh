// round2.cuh -- the second round of the lazy lists, launched from the device. Included by round2.cu only.
//
// The first blend phase parks the tiles whose list prefix ran out with a pixel still live. What they need then is
// the rest of the pipeline for the rest of the scene: the back of the depth order (front-first frames), its offsets,
// every record, the block entries behind the first slab, the rest of the parked tiles' lists, and the second blend
// phase. At the paper's kind of scene nothing parks (config 3, config 4: zero tiles), and launching those kernels from
// the host just to have each of them read a zero cost 25-35 us per frame. So the host launches one thread instead
// (r2_gate_kernel) that reads the parked count and, if it is not zero, launches them (r2_tail_launch): tail launches
// run in order after the launching grid has completed, and the stream's next operation waits for them. The host
// describes the launches in an R2Chain (blend.cuh) before the first phase.
#pragma once

#include "blend.cuh"
#include "blockbin.cuh"
#include "onesweep.cuh"
#include "preprocess.cuh"
#include "scan_dup.cuh"

namespace pvg {

template <int BITS>
__device__ __forceinline__ void r2_launch_emit(const R2Chain& c) {
  bin_emit_kernel<BITS, false><<<c.emit_grid, BP_THREADS, sizeof(BinEmitSmem<BITS>), cudaStreamTailLaunch>>>(
      c.nv, c.Mb, c.boffsets, c.chunk_owner, c.scan_keys, c.visit, c.blocks_x, c.s_g, c.s_mask, c.bin_start, c.emit_lookback,
      c.emit_ticket, nullptr, nullptr, c.emit_tiles);
}

template <bool COUNT, int MODE>
__device__ __noinline__ void r2_tail_launch(const FrameParams& P, const R2Chain& c, const uint2* ranges, const uint32_t* vals,
                                            const float4* record, float* out_rgb, float* out_depth, float* out_alpha,
                                            unsigned long long* counters, const float* featw, const BlendLazy& Z) {
  const cudaStream_t ts = cudaStreamTailLaunch;
  if (c.back) {
    depth_select_kernel<true><<<c.sel_grid, SEL_THREADS, 0, ts>>>(c.okeys, c.n, c.fc, c.sel_keys, c.sel_vals, nullptr, c.sel_region,
                                                                 c.sel_status, c.sel_ticket, c.sel_side, c.lb, c.lb_rows, c.lb_tile,
                                                                 nullptr);
    const DepthCtl* ctl = reinterpret_cast<const DepthCtl*>(c.sel_region + DH_CTL);
    uint64_t* lb = c.lb;
    for (uint32_t p = 0; p < c.passes; ++p) {
      const uint32_t* hist = c.sel_region + p * DS_RADIX;
      if (p < 3)
        depth_pass_kernel<PVG_DS_THREADS, PVG_DS_ITEMS, DS_BITS, PVG_DS_MINB, false, true>
            <<<c.pass_grid, PVG_DS_THREADS, sizeof(OnesweepSmem<PVG_DS_THREADS, PVG_DS_ITEMS, DS_BITS>), ts>>>(
                c.ka, c.va, c.kb, c.vb, c.back_count, (int)p, ds_shift((int)p), ctl, hist, lb, c.pass_tickets + p, nullptr);
      else
        depth_pass_kernel<PVG_DS_THREADS, PVG_DS_ITEMS, DS_TOP_BITS, PVG_DS_MINB, false, true>
            <<<c.pass_grid, PVG_DS_THREADS, sizeof(OnesweepSmem<PVG_DS_THREADS, PVG_DS_ITEMS, DS_TOP_BITS>), ts>>>(
                c.ka, c.va, c.kb, c.vb, c.back_count, (int)p, ds_shift((int)p), ctl, hist, lb, c.pass_tickets + p, nullptr);
      lb += (size_t)c.lb_rows << ds_bits((int)p);
    }
    scan_counts_kernel<true><<<c.scan_grid, SCAN_THREADS, 0, ts>>>(c.back_count, c.counts, c.scan_keys, c.visit, c.boffsets,
                                                                  c.scan_total, c.scan_status, c.scan_ticket, c.chunk_owner,
                                                                  c.owner_chunk, c.rank0, c.scan_init, nullptr);
  }
  if (c.shade)
    shade_all_kernel<<<c.shade_grid, 256, 0, ts>>>(P, c.n, c.counts, nullptr, c.A0, c.A1, c.A2, c.A3, c.SH, c.record, c.featw);
  if (c.emit) {
    switch (c.emit_bits) {
      case 1: r2_launch_emit<1>(c); break;
      case 2: r2_launch_emit<2>(c); break;
      case 3: r2_launch_emit<3>(c); break;
      case 4: r2_launch_emit<4>(c); break;
      case 5: r2_launch_emit<5>(c); break;
      case 6: r2_launch_emit<6>(c); break;
      case 7: r2_launch_emit<7>(c); break;
      default: r2_launch_emit<8>(c); break;
    }
  }
  bin_write_kernel<<<c.write_grid, BW_THREADS, 0, ts>>>(c.s_g, c.s_mask, c.bin_start, c.bin_start + 257, c.ranges, c.tiles_x, c.tiles_y,
                                                       c.blocks_x, c.chunk_cnt, c.write_ticket, c.vals, c.kin_lo, 0xFFFFFFFFu,
                                                       c.want_mask, c.want_count, nullptr, c.avail, 1u);
  blend_kernel<COUNT, MODE, 2><<<c.blend_grid, BLEND_THREADS, 0, ts>>>(P, ranges, vals, record, out_rgb, out_depth, out_alpha, counters,
                                                                      featw, Z);
}

// One thread. which = COUNT * 3 + MODE of the frame's blend.
__global__ void r2_gate_kernel(const __grid_constant__ FrameParams P, const __grid_constant__ R2Chain c, int which,
                               const uint2* ranges, const uint32_t* vals, const float4* record, float* out_rgb, float* out_depth,
                               float* out_alpha, unsigned long long* counters, const float* featw,
                               const __grid_constant__ BlendLazy Z) {
  // launched as a programmatic dependent of the first blend phase (pvg_r2_gate): the thread is resident before that
  // kernel ends and waits here for its completion, so the launch latency of the gate is off the frame's critical path
  asm volatile("griddepcontrol.wait;" ::: "memory");
  const uint32_t parked = *Z.unf_count;
  *Z.parked_host = parked;
  if (!parked) return;
  switch (which) {
    case 0: r2_tail_launch<false, 0>(P, c, ranges, vals, record, out_rgb, out_depth, out_alpha, counters, featw, Z); break;
    case 1: r2_tail_launch<false, 1>(P, c, ranges, vals, record, out_rgb, out_depth, out_alpha, counters, featw, Z); break;
    case 2: r2_tail_launch<false, 2>(P, c, ranges, vals, record, out_rgb, out_depth, out_alpha, counters, featw, Z); break;
    case 3: r2_tail_launch<true, 0>(P, c, ranges, vals, record, out_rgb, out_depth, out_alpha, counters, featw, Z); break;
    case 4: r2_tail_launch<true, 1>(P, c, ranges, vals, record, out_rgb, out_depth, out_alpha, counters, featw, Z); break;
    default: r2_tail_launch<true, 2>(P, c, ranges, vals, record, out_rgb, out_depth, out_alpha, counters, featw, Z); break;
  }
}

}  // namespace pvg
