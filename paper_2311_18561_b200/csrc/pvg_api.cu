// pvg_api.cu -- host side of the C ABI declared in include/pvg.h.
// Orchestrates the five stages on one CUDA stream; every step of the path runs in the
// kernels of this directory. No CPU fallback: CUDA errors surface as PVG_ERR_CUDA.

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/pvg.h"
#include "blend.cuh"
#include "blockbin.cuh"
#include "calib.cuh"
#include "common.cuh"
#include "expand.cuh"
#include "front_sort.cuh"
#include "onesweep.cuh"
#include "preprocess.cuh"
#include "ranges.cuh"
#include "scan_dup.cuh"
#include "tilebin.cuh"

using namespace pvg;

namespace {

thread_local char g_cuda_err[512] = "";
pvg_alloc_fn g_alloc = nullptr;
pvg_free_fn g_free = nullptr;
void* g_alloc_user = nullptr;

#define CU(expr)                                                                              \
  do {                                                                                        \
    cudaError_t e_ = (expr);                                                                  \
    if (e_ != cudaSuccess) {                                                                  \
      snprintf(g_cuda_err, sizeof(g_cuda_err), "%s:%d %s -> %s", __FILE__, __LINE__, #expr,   \
               cudaGetErrorString(e_));                                                       \
      return PVG_ERR_CUDA;                                                                    \
    }                                                                                         \
  } while (0)

#define TRY(expr)            \
  do {                       \
    int rc_ = (expr);        \
    if (rc_ != PVG_OK) return rc_; \
  } while (0)

// The first slab of the lazy lists holds at least this many halves of (blocks x LAZY_CHUNKS chunks x 512) entries
// (lazy_emit_first, common.cuh). Config 1 / config 2, ms per frame: 2 halves 0.2228 / 0.3151, 3: 0.2255 / 0.3107,
// 4: 0.2489 / 0.3300 (no tile parks with any; without a floor 800 of config 1's 2400 tiles park at a slab of 1/16).
#ifndef PVG_LAZY_FLOOR_HALVES
#define PVG_LAZY_FLOOR_HALVES 3
#endif
// PVG_OPT_LAZY_DEPTH = 1 (auto): front-first depth order for scenes of at least this many Gaussians. Its fixed costs (the
// selection's latency chain, one more launch) outweigh the sort it saves on small scenes: config 1 (200 k) 0.2255 ms per
// frame with it, 0.2046 without; config 2 (1 M) 0.313 / 0.333; config 3 (3 M) 0.292 / 0.380.
#ifndef PVG_LAZY_DEPTH_MIN_N
#define PVG_LAZY_DEPTH_MIN_N (1u << 19)
#endif

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: remember per (call site, device), thread-safe.
#define PVG_ENSURE_SMEM(kern, bytes, dev)                                                              \
  do {                                                                                                 \
    static std::atomic<uint64_t> done_[4];                                                             \
    const unsigned d_ = (unsigned)(dev) & 255u;                                                        \
    if (!(done_[d_ >> 6].load(std::memory_order_acquire) & (1ull << (d_ & 63u)))) {                    \
      CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(bytes)));       \
      done_[d_ >> 6].fetch_or(1ull << (d_ & 63u), std::memory_order_release);                          \
    }                                                                                                  \
  } while (0)

// The caller's current device for the duration of an entry point (a scene lives on the device it was created on).
struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) {
    int cur = -1;
    if (dev >= 0 && cudaGetDevice(&cur) == cudaSuccess && cur != dev && cudaSetDevice(dev) == cudaSuccess) prev = cur;
  }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

// device ordinal and SM count, looked up once (pvg_create_scene) instead of on every frame
struct Dev {
  int ordinal = 0, sms = 1, coop = 0;   // coop: cooperative launches supported (front_sort_kernel)
  int query() {
    CU(cudaGetDevice(&ordinal));
    CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, ordinal));
    CU(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, ordinal));
    return PVG_OK;
  }
};

// Guard bands (pvg_guard_bands / pvg_check_guards; a test hook: compute-sanitizer is not available on every pool): every
// device allocation of the library gets kGuard bytes of a known pattern in front and behind; a kernel that writes out
// of bounds of a workspace buffer by less than that damages a band, which pvg_check_guards finds.
constexpr size_t kGuard = 4096;
constexpr int kGuardByte = 0xA5;
std::atomic<bool> g_guards{false};
std::mutex g_guard_mu;
std::map<void*, size_t> g_guarded;   // user pointer -> user bytes

void* raw_alloc(size_t bytes, cudaStream_t st) {
  if (g_alloc) return g_alloc(bytes, (void*)st, g_alloc_user);
  void* p = nullptr;
  if (cudaMalloc(&p, bytes) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  return p;
}
void raw_free(void* p) {
  if (g_free) g_free(p, g_alloc_user);
  else cudaFree(p);
}
void* dev_alloc(size_t bytes, cudaStream_t st) {
  if (bytes == 0) bytes = 256;
  if (!g_guards.load()) return raw_alloc(bytes, st);
  bytes = (bytes + 255) & ~(size_t)255;
  unsigned char* base = static_cast<unsigned char*>(raw_alloc(bytes + 2 * kGuard, st));
  if (!base) return nullptr;
  if (cudaMemset(base, kGuardByte, kGuard) != cudaSuccess || cudaMemset(base + kGuard + bytes, kGuardByte, kGuard) != cudaSuccess) {
    cudaGetLastError();
    raw_free(base);
    return nullptr;
  }
  std::lock_guard<std::mutex> lk(g_guard_mu);
  g_guarded[base + kGuard] = bytes;
  return base + kGuard;
}
void dev_free(void* p) {
  if (!p) return;
  {
    std::lock_guard<std::mutex> lk(g_guard_mu);
    auto it = g_guarded.find(p);
    if (it != g_guarded.end()) {
      g_guarded.erase(it);
      p = static_cast<unsigned char*>(p) - kGuard;
    }
  }
  raw_free(p);
}

// growable device buffer
struct Buf {
  void* p = nullptr;
  size_t cap = 0;
  int reserve(size_t bytes, cudaStream_t st, double headroom = 1.0) {
    if (bytes <= cap) return PVG_OK;
    if (p) {
      // Growing a live buffer: a caching allocator (the torch hooks) would re-issue the block at once to work on the
      // stream it was allocated for, while kernels of this scene -- on its current, side or copy stream, possibly
      // another stream than the one of the allocation -- may still read it. Growth is rare (headroom): wait.
      cudaDeviceSynchronize();
      dev_free(p);
    }
    p = nullptr;
    cap = 0;
    size_t want = (size_t)((double)bytes * headroom);
    want = (want + 255) & ~(size_t)255;
    p = dev_alloc(want, st);
    if (!p && want > bytes) { want = (bytes + 255) & ~(size_t)255; p = dev_alloc(want, st); }
    if (!p) return PVG_ERR_OOM;
    cap = want;
    return PVG_OK;
  }
  void release() { dev_free(p); p = nullptr; cap = 0; }
  template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

struct KernelRec {
  const char* name;
  int stage;
  cudaEvent_t e0, e1;
};

// Two tile shapes of the onesweep pass: large tiles amortise the look-back for the
// instance sort, small ones give the n-key depth sort enough CTAs to fill 148 SMs.
#ifndef PVG_OSL_THREADS
#define PVG_OSL_THREADS 384
#define PVG_OSL_ITEMS 16
#define PVG_OSL_MINB 2
#endif
struct OsLarge { static constexpr int THREADS = PVG_OSL_THREADS, ITEMS = PVG_OSL_ITEMS, MINB = PVG_OSL_MINB; static constexpr bool STREAM = true; };
#ifndef PVG_OSS_THREADS
#define PVG_OSS_THREADS 256   // cfg 3 depth passes: 256 x 16 0.141 ms, 384 x 8 0.149, 256 x 24 0.146, 512 x 8 0.154, 256 x 8 (3 CTAs/SM) 0.158
#define PVG_OSS_ITEMS 16
#define PVG_OSS_MINB 2
#endif
struct OsSmall { static constexpr int THREADS = PVG_OSS_THREADS, ITEMS = PVG_OSS_ITEMS, MINB = PVG_OSS_MINB; static constexpr bool STREAM = false; };
#ifndef PVG_OS_SMALL_BELOW
#define PVG_OS_SMALL_BELOW (8u << 20)
#endif
constexpr uint64_t OS_SMALL_BELOW = PVG_OS_SMALL_BELOW;

// scratch of one sort call
// layout of pvg_scene::unf: [256] u64 block masks | u32 parked count (+ pad) | [tiles] u32 lim | [tiles] u32 parked list
constexpr size_t kUnfHead = 2048 + 64;
constexpr size_t kDhistWords = DH_WORDS;   // 4 x 512 digit counts, the CTA counter and the depth sort's control block

struct SortScratch {
  Buf hist;      // [passes][256] u32
  Buf lookback;  // [passes][tiles][256] u64
  Buf tickets;   // [passes] u32
};

struct Timer {
  bool enabled = false;      // PVG_OPT_KERNEL_EVENTS (default off: a measurement hook)
  bool accumulate = false;  // keep the records of every frame until they are read
  int stride = 1;           // record the launches of every stride-th render only (PVG_OPT_EVENT_STRIDE)
  uint64_t renders = 0;     // renders since the options were last set
  bool frame_on = true;     // this render records
  void next_frame() { frame_on = enabled && (renders++ % (uint64_t)stride == 0); }
  std::vector<KernelRec> recs;     // launches of the current frame
  std::vector<cudaEvent_t> pool;   // reusable events
  size_t used = 0;
  int get(cudaEvent_t* e) {
    if (used == pool.size()) {
      cudaEvent_t ev;
      CU(cudaEventCreate(&ev));
      pool.push_back(ev);
    }
    *e = pool[used++];
    return PVG_OK;
  }
  // Back-to-back kernels of one stream share their boundary event (the end of one is the start of the next):
  // every event record between two kernels costs ~2 us of stream time, 28 records were 5% of a 1 ms frame.
  // A shared start includes the ~1 us launch gap in the next kernel's time. Anything else enqueued on the
  // stream (a wait on another stream, a memset, a copy) must call cut() so that it is not billed to a kernel.
  cudaStream_t chain_stream = nullptr;
  cudaEvent_t chain_event = nullptr;
  // programmatic dependent launch: the last operation enqueued on pdl_stream was a kernel of the chain (launch_chain);
  // anything else -- a memset, an event, a wait, a copy: whatever calls cut(), or an event record of this timer -- breaks it
  cudaStream_t pdl_stream = nullptr;
  bool pdl_open = false;
  void cut() { chain_event = nullptr; pdl_open = false; }
  void reset() { recs.clear(); used = 0; cut(); }
  int begin(const char* name, int stage, cudaStream_t st) {
    if (!frame_on) return PVG_OK;
    KernelRec r{name, stage, nullptr, nullptr};
    pdl_open = false;
    if (chain_event && chain_stream == st) {
      r.e0 = chain_event;
    } else {
      TRY(get(&r.e0));
      CU(cudaEventRecord(r.e0, st));
    }
    TRY(get(&r.e1));
    recs.push_back(r);
    return PVG_OK;
  }
  int end(cudaStream_t st) {
    if (!frame_on) return PVG_OK;
    CU(cudaEventRecord(recs.back().e1, st));
    pdl_open = false;
    chain_stream = st;
    chain_event = recs.back().e1;
    return PVG_OK;
  }
  void destroy() {
    for (cudaEvent_t e : pool) cudaEventDestroy(e);
    pool.clear();
    recs.clear();
    used = 0;
  }
};

// Launch of a kernel of the frame's main chain (they all begin with pdl_launch_dependents(); pdl_wait();): as a
// programmatic dependent of the previous kernel when that one was the last thing enqueued on the stream, so that its
// launch latency and its CTAs' start overlap the previous kernel's tail (PVG_PDL=0: always plain launches).
#ifndef PVG_PDL
#define PVG_PDL 1
#endif
template <class... KArgs, class... Args>
int launch_chain(Timer* tm, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = (PVG_PDL && tm && tm->pdl_open && tm->pdl_stream == st) ? 1 : 0;
  CU(cudaLaunchKernelEx(&cfg, kern, KArgs(args)...));
  if (tm) { tm->pdl_open = true; tm->pdl_stream = st; }
  return PVG_OK;
}

template <class Cfg, int BITS, int HI>
int launch_pass_bits(const uint64_t* kin, const uint32_t* vin, uint64_t* kout, uint32_t* vout, uint32_t n, int shift,
                     const uint32_t* hist, uint64_t* lookback, uint32_t* ticket, cudaStream_t st, int dev) {
  using Smem = OnesweepSmem<Cfg::THREADS, Cfg::ITEMS, BITS>;
  auto kern = onesweep_pass_kernel<Cfg::THREADS, Cfg::ITEMS, BITS, Cfg::MINB, HI, Cfg::STREAM>;
  PVG_ENSURE_SMEM(kern, sizeof(Smem), dev);
  constexpr uint32_t TILE = Cfg::THREADS * Cfg::ITEMS;
  const uint32_t tiles = (n + TILE - 1) / TILE;
  kern<<<tiles, Cfg::THREADS, sizeof(Smem), st>>>(kin, vin, kout, vout, n, shift & 31, hist, lookback, ticket);
  return PVG_OK;
}

template <class Cfg>
int launch_pass(int bits, const uint64_t* kin, const uint32_t* vin, uint64_t* kout, uint32_t* vout, uint32_t n, int shift,
                const uint32_t* hist, uint64_t* lookback, uint32_t* ticket, cudaStream_t st, int dev) {
  switch (bits) {
#define PVG_CASE(B)                                                                                              \
  case B:                                                                                                        \
    return shift >= 32 ? launch_pass_bits<Cfg, B, 1>(kin, vin, kout, vout, n, shift, hist, lookback, ticket, st, dev) \
                       : launch_pass_bits<Cfg, B, 0>(kin, vin, kout, vout, n, shift, hist, lookback, ticket, st, dev);
    PVG_CASE(1) PVG_CASE(2) PVG_CASE(3) PVG_CASE(4) PVG_CASE(5) PVG_CASE(6) PVG_CASE(7) PVG_CASE(8)
#undef PVG_CASE
    default: return PVG_ERR_BAD_OPTION;
  }
}

// Stable LSD sort of n pairs on key bits [begin_bit, end_bit). Buffers ping-pong; *result
// tells which side (0: a, 1: b) holds the sorted list.
// Sizes and zeroes the scratch of one sort call (histograms, tickets, look-back words) on stream zs -- the
// renderer does this on its side stream while preprocess runs, so the memsets are off the critical path.
int prep_onesweep(uint64_t n, int begin_bit, int end_bit, cudaStream_t alloc_st, cudaStream_t zs, SortScratch& sc,
                  bool hist_ready) {
  if (n == 0 || end_bit <= begin_bit) return PVG_OK;
  const SortPlan plan = make_sort_plan(begin_bit, end_bit);
  const bool small = n < OS_SMALL_BELOW;
  const uint64_t tile_sz = small ? OsSmall::THREADS * OsSmall::ITEMS : OsLarge::THREADS * OsLarge::ITEMS;
  const uint64_t tiles = (n + tile_sz - 1) / tile_sz;
  TRY(sc.hist.reserve((size_t)OS_MAX_PASSES * OS_RADIX * 4, alloc_st));
  TRY(sc.tickets.reserve((size_t)OS_MAX_PASSES * 4, alloc_st));
  TRY(sc.lookback.reserve((size_t)plan.num_passes * tiles * OS_RADIX * 8, alloc_st, 1.25));
  if (!hist_ready) CU(cudaMemsetAsync(sc.hist.p, 0, (size_t)OS_MAX_PASSES * OS_RADIX * 4, zs));
  CU(cudaMemsetAsync(sc.tickets.p, 0, (size_t)OS_MAX_PASSES * 4, zs));
  CU(cudaMemsetAsync(sc.lookback.p, 0, (size_t)plan.num_passes * tiles * OS_RADIX * 8, zs));
  return PVG_OK;
}

int run_onesweep(const Dev& dv, uint64_t n, uint64_t* ka, uint32_t* va, uint64_t* kb, uint32_t* vb, int begin_bit,
                 int end_bit, cudaStream_t st, SortScratch& sc, Timer* tm, int stage, int* result,
                 bool hist_ready = false, bool scratch_ready = false, const uint32_t* hist_at = nullptr) {
  *result = 0;
  if (n == 0 || end_bit <= begin_bit) return PVG_OK;
  const SortPlan plan = make_sort_plan(begin_bit, end_bit);
  const bool small = n < OS_SMALL_BELOW;
  const uint64_t tile_sz = small ? OsSmall::THREADS * OsSmall::ITEMS : OsLarge::THREADS * OsLarge::ITEMS;
  const uint64_t tiles = (n + tile_sz - 1) / tile_sz;
  if (!scratch_ready) {
    TRY(prep_onesweep(n, begin_bit, end_bit, st, st, sc, hist_ready));
    if (tm) tm->cut();
  }

  const uint64_t hist_chunks = (n + (uint64_t)HIST_THREADS * HIST_ITEMS - 1) / ((uint64_t)HIST_THREADS * HIST_ITEMS);
  const unsigned hist_grid = (unsigned)std::min<uint64_t>(hist_chunks, (uint64_t)dv.sms * 4);
  if (!hist_ready) {
    if (tm) TRY(tm->begin("onesweep_histogram", stage, st));
    uint32_t* done = sc.tickets.as<uint32_t>() + (OS_MAX_PASSES - 1);   // last ticket slot: never a pass's (<= 8 passes)
    if (small) onesweep_histogram_kernel<false><<<hist_grid, HIST_THREADS, 0, st>>>(ka, n, plan, sc.hist.as<uint32_t>(), done);
    else onesweep_histogram_kernel<true><<<hist_grid, HIST_THREADS, 0, st>>>(ka, n, plan, sc.hist.as<uint32_t>(), done);
    if (tm) TRY(tm->end(st));
  }

  uint64_t* kin = ka; uint32_t* vin = va; uint64_t* kout = kb; uint32_t* vout = vb;
  for (int p = 0; p < plan.num_passes; ++p) {
    if (tm) TRY(tm->begin("onesweep_pass", stage, st));
    const uint32_t* hist = (hist_at ? hist_at : sc.hist.as<uint32_t>()) + p * OS_RADIX;
    uint64_t* lb = sc.lookback.as<uint64_t>() + (size_t)p * tiles * OS_RADIX;
    uint32_t* tk = sc.tickets.as<uint32_t>() + p;
    if (small) TRY(launch_pass<OsSmall>(plan.bits[p], kin, vin, kout, vout, (uint32_t)n, plan.shift[p], hist, lb, tk, st, dv.ordinal));
    else TRY(launch_pass<OsLarge>(plan.bits[p], kin, vin, kout, vout, (uint32_t)n, plan.shift[p], hist, lb, tk, st, dv.ordinal));
    if (tm) TRY(tm->end(st));
    std::swap(kin, kout);
    std::swap(vin, vout);
  }
  CU(cudaGetLastError());
  *result = plan.num_passes & 1;
  return PVG_OK;
}

// ---- the depth sort of the Gaussians (onesweep.cuh: 9 + 9 + 9 + 4 bits, pass 0 drops the culled pairs) ----------
struct DsCfg { static constexpr int THREADS = PVG_DS_THREADS, ITEMS = PVG_DS_ITEMS, MINB = PVG_DS_MINB; };
constexpr uint32_t kDsTile = DsCfg::THREADS * DsCfg::ITEMS;

inline size_t depth_lookback_words(uint32_t n) {
  const size_t tiles = (n + kDsTile - 1) / kDsTile;
  return tiles * (size_t)(3 * DS_RADIX + (1 << DS_TOP_BITS));
}

// The front of a front-first frame is small (tens of thousands of pairs): its passes run on small tiles, so that the
// few tiles spread over many SMs and a tile's latency -- which is all a pass costs at that size -- is short.
#ifndef PVG_DSF_THREADS
#define PVG_DSF_THREADS 512
#define PVG_DSF_ITEMS 2
#define PVG_DSF_MINB 2
#endif
struct DsFrontCfg { static constexpr int THREADS = PVG_DSF_THREADS, ITEMS = PVG_DSF_ITEMS, MINB = PVG_DSF_MINB; };
constexpr uint32_t kDsFrontTile = DsFrontCfg::THREADS * DsFrontCfg::ITEMS;
inline size_t class_lookback_rows(uint32_t n, int cls) { const uint32_t t = cls ? kDsTile : kDsFrontTile; return (n + t - 1) / t; }
inline size_t class_lookback_words(uint32_t n, int cls) { return class_lookback_rows(n, cls) * (size_t)(3 * DS_RADIX + (1 << DS_TOP_BITS)); }

// sizes and zeroes the tickets and look-back words of the four passes on stream zs
// front_first: the front's passes and the back's have their own tickets (0..3 / 4..7) and look-back words, and
// depth_select_kernel zeroes the words its class will use (it knows how many pairs there are)
int prep_depth_sort(uint32_t n, cudaStream_t alloc_st, cudaStream_t zs, SortScratch& sc, bool front_first = false) {
  static_assert(OS_MAX_PASSES >= 2 * DS_PASSES + 1, "tickets of two classes and the barrier word of front_sort_kernel");
  TRY(sc.tickets.reserve((size_t)OS_MAX_PASSES * 4, alloc_st));
  CU(cudaMemsetAsync(sc.tickets.p, 0, (size_t)OS_MAX_PASSES * 4, zs));
  if (front_first) {
    TRY(sc.lookback.reserve((class_lookback_words(n, 0) + class_lookback_words(n, 1)) * 8, alloc_st, 1.25));
  } else {
    TRY(sc.lookback.reserve(depth_lookback_words(n) * 8, alloc_st, 1.25));
    CU(cudaMemsetAsync(sc.lookback.p, 0, depth_lookback_words(n) * 8, zs));
  }
  return PVG_OK;
}

// loop_ctas > 0: a launch of at most that many CTAs that loop over tickets (the number of pairs is on the device)
template <int BITS, bool FIRST, bool LOOP = false, class Cfg = DsCfg>
int launch_depth_pass(uint64_t* ka, uint32_t* va, uint64_t* kb, uint32_t* vb, uint32_t n, int pass, const DepthCtl* ctl,
                      const uint32_t* hist, uint64_t* lookback, uint32_t* ticket, cudaStream_t st, int dev, Timer* tm,
                      unsigned loop_ctas = 0, const uint32_t* only_if = nullptr) {
  using Smem = OnesweepSmem<Cfg::THREADS, Cfg::ITEMS, BITS>;
  auto kern = depth_pass_kernel<Cfg::THREADS, Cfg::ITEMS, BITS, Cfg::MINB, FIRST, LOOP>;
  PVG_ENSURE_SMEM(kern, sizeof(Smem), dev);
  constexpr uint32_t TILE = Cfg::THREADS * Cfg::ITEMS;
  unsigned grid = (n + TILE - 1) / TILE;
  if (LOOP) grid = std::max(1u, std::min(grid, loop_ctas));
  return launch_chain(tm, kern, dim3(grid), dim3(Cfg::THREADS), sizeof(Smem), st, ka, va, kb, vb, n, pass,
                      ds_shift(pass), ctl, hist, lookback, ticket, only_if);
}

// dh: this frame's dhist half (exclusive digit prefixes + DepthCtl, written by preprocess). Every pass is launched
// for n pairs; passes 1..3 read S and their input side from the control block and exit at once if they are the identity.
// Launches passes [p0, p1). The frame launches 0..2 at once and the top-digit pass after its host wait, only if
// preprocess found it to be needed (it is the identity unless the far plane is beyond 65536 znear).
int run_depth_sort(const Dev& dv, uint32_t n, uint64_t* ka, uint32_t* va, uint64_t* kb, uint32_t* vb, const uint32_t* dh,
                   cudaStream_t st, SortScratch& sc, Timer* tm, int p0 = 0, int p1 = DS_PASSES) {
  const DepthCtl* ctl = reinterpret_cast<const DepthCtl*>(dh + DH_CTL);
  const size_t tiles = (n + kDsTile - 1) / kDsTile;
  uint64_t* lb = sc.lookback.as<uint64_t>();
  uint32_t* tk = sc.tickets.as<uint32_t>();
  for (int p = 0; p < p0; ++p) lb += tiles * (size_t)(1 << ds_bits(p));
  for (int p = p0; p < p1; ++p) {
    if (tm) TRY(tm->begin("onesweep_pass", PVG_STAGE_DEPTH_SORT, st));
    const uint32_t* hist = dh + p * DS_RADIX;
    if (p == 0) TRY((launch_depth_pass<DS_BITS, true>(ka, va, kb, vb, n, p, ctl, hist, lb, tk + p, st, dv.ordinal, tm)));
    else if (p < 3) TRY((launch_depth_pass<DS_BITS, false>(ka, va, kb, vb, n, p, ctl, hist, lb, tk + p, st, dv.ordinal, tm)));
    else TRY((launch_depth_pass<DS_TOP_BITS, false>(ka, va, kb, vb, n, p, ctl, hist, lb, tk + p, st, dv.ordinal, tm)));
    if (tm) TRY(tm->end(st));
    lb += tiles * (size_t)(1 << ds_bits(p));
  }
  CU(cudaGetLastError());
  return PVG_OK;
}

#ifndef PVG_CP_THREADS
#define PVG_CP_THREADS 384
#define PVG_CP_ITEMS 16
#define PVG_CP_MINB 2
#endif
struct CpCfg { static constexpr int THREADS = PVG_CP_THREADS, ITEMS = PVG_CP_ITEMS, MINB = PVG_CP_MINB; };

template <int BITS, bool LAST>
int launch_compact_bits(const uint16_t* tin, const uint32_t* vin, uint16_t* tout, uint32_t* vout, uint32_t n, int shift,
                        const uint32_t* hist, uint64_t* lookback, uint32_t* ticket, cudaStream_t st, int dev) {
  using Smem = CompactSmem<CpCfg::THREADS, CpCfg::ITEMS, BITS>;
  auto kern = compact_pass_kernel<CpCfg::THREADS, CpCfg::ITEMS, BITS, CpCfg::MINB, LAST>;
  PVG_ENSURE_SMEM(kern, sizeof(Smem), dev);
  constexpr uint32_t TILE = CpCfg::THREADS * CpCfg::ITEMS;
  kern<<<(n + TILE - 1) / TILE, CpCfg::THREADS, sizeof(Smem), st>>>(tin, vin, tout, vout, n, shift, hist, lookback, ticket);
  return PVG_OK;
}

// Tile-id passes over the compact (u16 tile, u32 index) payload; histograms come from
// tile_prefix_kernel. The sorted indices end in v[*result]; t[] ping-pongs alongside.
int run_compact_sort(const Dev& dv, uint32_t n, uint16_t* t0, uint32_t* v0, uint16_t* t1, uint32_t* v1, int tile_bits, cudaStream_t st,
                     SortScratch& sc, Timer* tm, int* result) {
  *result = 0;
  if (n == 0) return PVG_OK;
  const SortPlan plan = make_sort_plan(32, 32 + tile_bits);
  constexpr uint64_t TILE = CpCfg::THREADS * CpCfg::ITEMS;
  const uint64_t tiles = (n + TILE - 1) / TILE;
  TRY(sc.tickets.reserve((size_t)OS_MAX_PASSES * 4, st));
  TRY(sc.lookback.reserve((size_t)plan.num_passes * tiles * OS_RADIX * 8, st, 1.25));
  CU(cudaMemsetAsync(sc.tickets.p, 0, (size_t)OS_MAX_PASSES * 4, st));
  CU(cudaMemsetAsync(sc.lookback.p, 0, (size_t)plan.num_passes * tiles * OS_RADIX * 8, st));
  if (tm) tm->cut();
  uint16_t* tin = t0; uint32_t* vin = v0; uint16_t* tout = t1; uint32_t* vout = v1;
  for (int p = 0; p < plan.num_passes; ++p) {
    const bool last = p == plan.num_passes - 1;
    const uint32_t* hist = sc.hist.as<uint32_t>() + p * OS_RADIX;
    uint64_t* lb = sc.lookback.as<uint64_t>() + (size_t)p * tiles * OS_RADIX;
    uint32_t* tk = sc.tickets.as<uint32_t>() + p;
    const int shift = plan.shift[p] - 32;
    if (tm) TRY(tm->begin(last ? "compact_pass_last" : "compact_pass", PVG_STAGE_SORT, st));
    int rc = PVG_ERR_BAD_OPTION;
    switch (plan.bits[p]) {
#define PVG_CASE(B)                                                                                   \
  case B:                                                                                             \
    rc = last ? launch_compact_bits<B, true>(tin, vin, tout, vout, n, shift, hist, lb, tk, st, dv.ordinal)   \
              : launch_compact_bits<B, false>(tin, vin, tout, vout, n, shift, hist, lb, tk, st, dv.ordinal); \
    break;
      PVG_CASE(1) PVG_CASE(2) PVG_CASE(3) PVG_CASE(4) PVG_CASE(5) PVG_CASE(6) PVG_CASE(7) PVG_CASE(8)
#undef PVG_CASE
      default: break;
    }
    TRY(rc);
    if (tm) TRY(tm->end(st));
    std::swap(tin, tout);
    std::swap(vin, vout);
  }
  CU(cudaGetLastError());
  *result = plan.num_passes & 1;
  return PVG_OK;
}

}  // namespace

// The re-laid-out model (SoA, preprocess.cuh), shared by a scene and its forks (pvg_fork_scene).
struct Model {
  Buf A0, A1, A2, A3, SH, shflag;
  std::atomic<int> refs{1};
};

struct pvg_scene {
  uint32_t n = 0;
  uint32_t nv = 0;   // pairs in visiting order that take part in the last frame: the S survivors (PRESORT_DEPTH) or n
  float cycle = 0.2f;
  int sh_degree = 3;
  cudaStream_t stream = nullptr;
  cudaEvent_t ev_switch = nullptr;    // orders a new stream (pvg_set_stream) behind the work still in flight on the old one
  Dev dev;                            // the device the scene lives on
  // options
  int presort = 1, keep_unsorted = 0, count_pairs = 0, compact = 1, block = 1, blend_cull = 1;
  int band_begin = 0, band_end = 0;   // PVG_OPT_TILE_ROW_BEGIN / END (0, 0: the whole image)
  int lazy_chunks = 2;                // PVG_OPT_LAZY_CHUNKS (0: always write the complete lists)
  // PVG_OPT_LAZY_SLAB: the first 1/lazy_slab of the block entries is emitted up front. B200, ms per frame of the config 3
  // sweep / config 4 (no tile parks at any of these): 4: 0.369 / 0.679, 8: 0.338 / 0.667, 12: 0.304 / 0.659,
  // 16: 0.300 / 0.659, 24: 0.304 / 0.648, 32: 0.302 / 0.646 -- the front the frame orders, scans and shades shrinks
  // with the slab (36 k Gaussians at 8, 16 k at 16); beyond 16 nothing is left to gain and parking comes closer
  int lazy_slab = 16;
  int exact_tiles = 0;                // PVG_OPT_EXACT_TILES: list a Gaussian only in the tiles its ellipse can reach (P13)
  int lazy_depth = 1;                 // PVG_OPT_LAZY_DEPTH: with lazy lists, order the front of the scene first (onesweep.cuh); 1: auto (large scenes), 2: always
  bool front_used = false;            // the last frame ordered its front first
  bool depth_complete = true;         // dvals[visit_side] holds all S survivors in depth order (pvg_debug_view completes it)
  uint64_t prev_parked = 0;           // tiles the frame before this one parked (read at this frame's host wait)
  uint32_t front = 0;                 // F: the pairs in front of the threshold
  int top_front = 0, top_back = 0;    // the class has keys of 2^27 and beyond
  Buf front_idx;                      // front-first: the front's Gaussian indices once more, for shade_list_kernel
  Buf okeys;                          // front-first: the n depth pairs of preprocess, index order (the sort's buffers ping-pong)
  Buf dsel;                           // front-first: 2 histogram regions (front, back) + 2 tickets
  Buf sel_status;                     // front-first: 2 x [tiles] look-back words of depth_select_kernel
  bool exact_used = false;            // the last frame built exact lists
  Buf tile_count, counts_exact;       // exact lists: per-tile and per-Gaussian counts of the refined masks
  uint32_t emit_first = 0, emit_tiles = 0, emit_radix = 256;   // bin_emit tiles in the first launch / in all; its look-back row length
  const uint32_t* visit_last = nullptr;
  bool visit_tail_done = false;       // pvg_debug_view has appended the culled Gaussians to the visiting order
  bool light = false;                 // this frame's preprocess left the records to shade_kernel
  bool records_complete = true;       // record[] holds every Gaussian's record (pvg_debug_view completes them on demand)
  float* featw_last = nullptr;
  // the option values the last render ran with: pvg_debug_view completes THAT frame, whatever was set since
  int presort_used = 1, keep_unsorted_used = 0, lazy_chunks_used = 0;
  bool lazy_used = false;             // last frame wrote list prefixes + what the unfinished tiles needed
  bool lists_complete = true;         // vals[] holds every tile's whole list (pvg_debug_view completes them on demand)
  bool compact_used = false;  // last frame carried (u16 tile, u32 index) instances
  bool block_used = false;    // last frame built the tile lists from 8x8-tile block entries (blockbin.cuh)
  Model* model = nullptr;
  // per-Gaussian workspace
  Buf record, tileinfo, counts, offsets, dkeys[2], dvals[2], scan_status, small;  // small: ticket u32 @0, total u64 @8
  // per-instance workspace
  Buf keys[2], vals[2], keys_unsorted, vals_unsorted;
  Buf tiles16[2], tiles16_unsorted;
  // block-entry workspace (blockbin.cuh)
  Buf boffsets, chunk_owner, e_bin, e_g, e_mask, s_g, s_mask, bin_tables, chunk_cnt;
  Buf lazy_state, unf;   // blend state of parked tiles [5][H W]; unfinished flags: [256] u64 block masks, then [tiles] u32
  Buf dhist;          // 2 x DH_WORDS u32 (preprocess.cuh): digit histograms + control block of the depth sort, double-buffered
  int dhist_side = 0;
  Buf ranges, tilegrid;
  Buf featw;   // clamp(rho, 0, 2) per Gaussian (dynamics target)
  Buf sky;     // cube map [6][res][res][3] (pvg_set_sky)
  int sky_res = 0;
  Buf img[2];  // render_host device images (double-buffered: the copy of frame k overlaps frame k + 1)
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t ev_rendered = nullptr, ev_copied[2] = {nullptr, nullptr};
  bool copy_pending[2] = {false, false};
  int img_next = 0;
  SortScratch sort_n, sort_m;
  uint64_t* h_total = nullptr;  // pinned, mapped
  uint64_t* d_total = nullptr;  // device alias of h_total (tile_prefix_kernel stores the totals through it)
  cudaStream_t side = nullptr;  // tile grid + prefix run here, beside the depth sort
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr, ev_start = nullptr, ev_zero = nullptr, ev_pre = nullptr;
  cudaStream_t aux = nullptr;   // front-first: the front's records are formed here, beside the sort and the tile grid
  cudaEvent_t ev_sel = nullptr, ev_aux = nullptr, ev_blocks = nullptr;
  Timer timer;
  // last frame
  uint64_t M = 0, Mb = 0, survivors = 0;
  FrameParams last_P{};
  int sorted_side = 0, visit_side = 0;
  uint32_t tiles_x = 0, tiles_y = 0;
  int sort_begin = 0, sort_end = 0;
  bool rendered = false;
};

namespace {

int ceil_log2(uint32_t v) {
  int b = 0;
  while ((1ull << b) < v) ++b;
  return b;
}

void release_all(pvg_scene* s) {
  if (s->model && s->model->refs.fetch_sub(1) == 1) {
    Buf* mb[] = {&s->model->A0, &s->model->A1, &s->model->A2, &s->model->A3, &s->model->SH, &s->model->shflag};
    for (Buf* b : mb) b->release();
    delete s->model;
  }
  s->model = nullptr;
  Buf* bufs[] = {&s->record, &s->tileinfo, &s->counts, &s->offsets,
                 &s->dkeys[0], &s->dkeys[1], &s->dvals[0], &s->dvals[1], &s->scan_status, &s->small,
                 &s->keys[0], &s->keys[1], &s->vals[0], &s->vals[1], &s->keys_unsorted, &s->vals_unsorted, &s->tiles16[0], &s->tiles16[1], &s->tiles16_unsorted,
                 &s->lazy_state, &s->unf, &s->dhist, &s->boffsets, &s->chunk_owner, &s->e_bin, &s->e_g, &s->e_mask, &s->s_g, &s->s_mask, &s->bin_tables, &s->chunk_cnt,
                 &s->tile_count, &s->counts_exact, &s->okeys, &s->front_idx, &s->dsel, &s->sel_status, &s->ranges, &s->tilegrid, &s->featw, &s->sky, &s->img[0], &s->img[1], &s->sort_n.hist, &s->sort_n.lookback, &s->sort_n.tickets,
                 &s->sort_m.hist, &s->sort_m.lookback, &s->sort_m.tickets};
  for (Buf* b : bufs) b->release();
  if (s->h_total) cudaFreeHost(s->h_total);
  s->h_total = nullptr;
  if (s->ev_switch) cudaEventDestroy(s->ev_switch);
  s->ev_switch = nullptr;
  if (s->ev_fork) cudaEventDestroy(s->ev_fork);
  if (s->ev_join) cudaEventDestroy(s->ev_join);
  if (s->ev_start) cudaEventDestroy(s->ev_start);
  if (s->ev_zero) cudaEventDestroy(s->ev_zero);
  if (s->ev_pre) cudaEventDestroy(s->ev_pre);
  s->ev_pre = nullptr;
  if (s->ev_sel) cudaEventDestroy(s->ev_sel);
  if (s->ev_aux) cudaEventDestroy(s->ev_aux);
  if (s->ev_blocks) cudaEventDestroy(s->ev_blocks);
  s->ev_sel = s->ev_aux = s->ev_blocks = nullptr;
  if (s->aux) cudaStreamDestroy(s->aux);
  s->aux = nullptr;
  s->ev_start = s->ev_zero = nullptr;
  if (s->side) cudaStreamDestroy(s->side);
  if (s->copy_stream) cudaStreamDestroy(s->copy_stream);
  if (s->ev_rendered) cudaEventDestroy(s->ev_rendered);
  for (int k = 0; k < 2; ++k) if (s->ev_copied[k]) cudaEventDestroy(s->ev_copied[k]);
  s->copy_stream = nullptr; s->ev_rendered = nullptr; s->ev_copied[0] = s->ev_copied[1] = nullptr;
  s->ev_fork = s->ev_join = nullptr;
  s->side = nullptr;
  s->timer.destroy();
}

int upload(Buf& dst, const float* src, size_t bytes, bool on_device, cudaStream_t st) {
  TRY(dst.reserve(bytes, st));
  CU(cudaMemcpyAsync(dst.p, src, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
  return PVG_OK;
}

int init_workspace(pvg_scene* s);

int create_impl(const pvg_scene_desc* d, pvg_scene* s) {
  int ndev = 0;
  CU(cudaGetDeviceCount(&ndev));
  if (ndev <= 0) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
    return PVG_ERR_CUDA;
  }
  TRY(s->dev.query());
  const size_t n = (size_t)d->n;
  s->n = (uint32_t)n;
  s->cycle = d->cycle;
  s->sh_degree = d->sh_degree;
  cudaStream_t st = s->stream;
  const bool dev = d->pointers_on_device != 0;
  Buf t_mu, t_quat, t_scale, t_op, t_sh, t_tau, t_beta, t_vel;
  int rc = PVG_OK;
  auto up = [&](Buf& b, const float* src, size_t floats) {
    if (rc == PVG_OK) rc = upload(b, src, floats * n * 4, dev, st);
  };
  up(t_mu, d->mu, 3); up(t_quat, d->quat, 4); up(t_scale, d->scale, 3); up(t_op, d->opacity, 1);
  up(t_sh, d->sh, 48); up(t_tau, d->tau, 1); up(t_beta, d->beta, 1); up(t_vel, d->vel, 3);
  auto rs = [&](Buf& b, size_t bytes) { if (rc == PVG_OK) rc = b.reserve(bytes, st); };
  s->model = new (std::nothrow) Model();
  if (!s->model) return PVG_ERR_OOM;
  Model* m = s->model;
  rs(m->A0, n * 16); rs(m->A1, n * 16); rs(m->A2, n * 16); rs(m->A3, n * 16); rs(m->SH, n * 192); rs(m->shflag, n);
  if (rc == PVG_OK) {
    relayout_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(
        (uint32_t)n, t_mu.as<float>(), t_quat.as<float>(), t_scale.as<float>(), t_op.as<float>(), t_sh.as<float>(),
        t_tau.as<float>(), t_beta.as<float>(), t_vel.as<float>(), m->A0.as<float4>(), m->A1.as<float4>(),
        m->A2.as<float4>(), m->A3.as<float4>(), m->SH.as<float4>(), m->shflag.as<uint8_t>());
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) {
      snprintf(g_cuda_err, sizeof(g_cuda_err), "relayout: %s", cudaGetErrorString(e));
      rc = PVG_ERR_CUDA;
    }
  }
  Buf* tmp[] = {&t_mu, &t_quat, &t_scale, &t_op, &t_sh, &t_tau, &t_beta, &t_vel};
  for (Buf* b : tmp) b->release();
  if (rc != PVG_OK) return rc;
  return init_workspace(s);
}

// The per-scene workspace (sized by n), streams and events: everything a scene or a fork owns besides the model.
int init_workspace(pvg_scene* s) {
  const size_t n = s->n;
  cudaStream_t st = s->stream;
  int rc = PVG_OK;
  auto rs = [&](Buf& b, size_t bytes) { if (rc == PVG_OK) rc = b.reserve(bytes, st); };
  rs(s->record, n * 48); rs(s->tileinfo, n * 16); rs(s->counts, n * 4); rs(s->offsets, n * 4); rs(s->boffsets, n * 4);
  rs(s->dkeys[0], n * 8); rs(s->dkeys[1], n * 8); rs(s->dvals[0], n * 4); rs(s->dvals[1], n * 4);
  rs(s->scan_status, ((n + SCAN_TILE - 1) / SCAN_TILE) * 16); rs(s->small, 256);
  rs(s->dhist, 2 * kDhistWords * 4);
  if (rc != PVG_OK) return rc;
  CU(cudaMemsetAsync(s->dhist.p, 0, 2 * kDhistWords * 4, st));
  CU(cudaStreamSynchronize(st));   // the first render may run on another stream: the zeroes must have landed
  CU(cudaEventCreateWithFlags(&s->ev_switch, cudaEventDisableTiming));
  CU(cudaHostAlloc((void**)&s->h_total, 128, cudaHostAllocMapped));
  memset(s->h_total, 0, 128);
  CU(cudaHostGetDevicePointer((void**)&s->d_total, s->h_total, 0));
  CU(cudaStreamCreateWithFlags(&s->side, cudaStreamNonBlocking));
  CU(cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming));
  CU(cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming));
  CU(cudaEventCreateWithFlags(&s->ev_start, cudaEventDisableTiming));
  CU(cudaEventCreateWithFlags(&s->ev_zero, cudaEventDisableTiming));
  CU(cudaEventCreateWithFlags(&s->ev_pre, cudaEventDisableTiming));
  CU(cudaEventCreateWithFlags(&s->ev_sel, cudaEventDisableTiming));
  CU(cudaEventCreateWithFlags(&s->ev_aux, cudaEventDisableTiming));
  CU(cudaEventCreateWithFlags(&s->ev_blocks, cudaEventDisableTiming));
  CU(cudaStreamCreateWithFlags(&s->aux, cudaStreamNonBlocking));
  CU(cudaStreamCreateWithFlags(&s->copy_stream, cudaStreamNonBlocking));
  CU(cudaEventCreateWithFlags(&s->ev_rendered, cudaEventDisableTiming));
  for (int k = 0; k < 2; ++k) CU(cudaEventCreateWithFlags(&s->ev_copied[k], cudaEventDisableTiming));
  return PVG_OK;
}

int fill_frame(const pvg_scene* s, const pvg_camera* cam, const pvg_state* state, FrameParams* P) {
  if (cam->width <= 0 || cam->height <= 0 || cam->width > 32768 || cam->height > 32768) return PVG_ERR_BAD_CAMERA;
  if (!(cam->fx > 0.f) || !(cam->fy > 0.f) || !std::isfinite(cam->fx) || !std::isfinite(cam->fy) ||
      !std::isfinite(cam->cx) || !std::isfinite(cam->cy))
    return PVG_ERR_BAD_CAMERA;
  for (int i = 0; i < 12; ++i)
    if (!std::isfinite(cam->world_to_cam[i])) return PVG_ERR_BAD_CAMERA;
  const float* E = cam->world_to_cam;
  for (int r = 0; r < 3; ++r) {
    for (int c = 0; c < 3; ++c) P->R[3 * r + c] = E[4 * r + c];
    P->T[r] = E[4 * r + 3];
  }
  for (int j = 0; j < 3; ++j)
    P->campos[j] = (float)-((double)E[j] * E[3] + (double)E[4 + j] * E[7] + (double)E[8 + j] * E[11]);
  P->fx = cam->fx; P->fy = cam->fy; P->cx = cam->cx; P->cy = cam->cy;
  for (int k = 0; k < 9; ++k) P->Rd[k] = (double)P->R[k];
  for (int k = 0; k < 3; ++k) P->Td[k] = (double)P->T[k];
  P->fxd = cam->fx; P->fyd = cam->fy; P->cxd = cam->cx; P->cyd = cam->cy;
  P->limx = (float)(1.3 * cam->width / (2.0 * (double)cam->fx));
  P->limy = (float)(1.3 * cam->height / (2.0 * (double)cam->fy));
  P->limxd = 1.3 * cam->width / (2.0 * (double)cam->fx);
  P->limyd = 1.3 * cam->height / (2.0 * (double)cam->fy);
  P->znear = cam->znear > 0.f ? cam->znear : PVG_ZNEAR_DEFAULT;
  P->t1 = (double)state->t - (double)state->dt;
  P->dts = state->dt;
  P->rho_min = state->rho_min;
  P->rho_max = state->rho_max;
  P->filter = (state->rho_min > 0.f || state->rho_max < INFINITY) ? 1 : 0;
  P->target = state->target;
  P->cull = s->blend_cull;
  P->linear = std::isinf(s->cycle) ? 1 : 0;
  P->inv_l = P->linear ? 0.f : (float)(1.0 / (double)s->cycle);
  P->inv_l_d = P->linear ? 0.0 : 1.0 / (double)s->cycle;
  P->two_over_l = P->linear ? 0.0 : 2.0 / (double)s->cycle;
  P->l_over_2pi = P->linear ? 0.0 : (double)s->cycle / (2.0 * 3.14159265358979323846);
  P->sh_degree = s->sh_degree;
  P->width = cam->width; P->height = cam->height;
  P->tiles_x = (cam->width + PVG_TILE - 1) / PVG_TILE;
  P->tiles_y = (cam->height + PVG_TILE - 1) / PVG_TILE;
  P->pack_rect = (P->tiles_x <= 256 && P->tiles_y <= 256) ? 1 : 0;
  P->band_y0 = s->band_begin;
  P->band_y1 = (s->band_end <= 0 || s->band_end > P->tiles_y) ? P->tiles_y : s->band_end;
  if (P->band_y0 >= P->band_y1) return PVG_ERR_BAD_STATE;
  for (int j = 0; j < 3; ++j) P->bg[j] = cam->bg[j];
  P->sky = s->sky_res > 0 ? s->sky.as<float>() : nullptr;
  P->sky_res = s->sky_res;
  P->lazy_slab = s->lazy_slab;
  {
    const uint64_t nb = (uint64_t)bb_blocks(P->tiles_x) * bb_blocks(P->tiles_y);
    P->lazy_min_tiles = (uint32_t)std::min<uint64_t>(((uint64_t)PVG_LAZY_FLOOR_HALVES * nb / 2 * (uint64_t)std::max(s->lazy_chunks, 0) * BB_CHUNK + PVG_EMIT_TILE - 1) / PVG_EMIT_TILE, 1u << 30);
  }
  return PVG_OK;
}

// PVG_BIN_FUSED=1: bin_emit_kernel forms the entries inside the split (no e_* round trip through HBM);
// 0: bin_expand_kernel + bin_pass_kernel.
#ifndef PVG_BIN_FUSED
#define PVG_BIN_FUSED 1
#endif
constexpr uint32_t kOwnerChunk = PVG_BIN_FUSED ? (uint32_t)BF_TILE : (uint32_t)BE_CHUNK;   // granularity of chunk_owner[]

// a2 scan of the per-Gaussian item counts in visiting order; the total lands in small @8.
// (the status words are there twice, and a second ticket and total at small @96 / @104: the front-first depth order
// scans the back of the visiting order in a launch of its own)
int prep_scan(pvg_scene* s, cudaStream_t zs) {
  const uint32_t scan_tiles = (s->n + SCAN_TILE - 1) / SCAN_TILE;
  CU(cudaMemsetAsync(s->scan_status.p, 0, (size_t)scan_tiles * 16, zs));
  CU(cudaMemsetAsync(s->small.p, 0, 16, zs));
  CU(cudaMemsetAsync(s->small.as<unsigned char>() + 96, 0, 16, zs));
  return PVG_OK;
}

// nv: the first nv visiting positions are scanned (the survivors after the depth sort; n otherwise)
// rank0 > 0 (blocks only): the second part of a front-first frame -- positions [rank0, rank0 + nv), continuing from the
// total the first part left; only_if: a device word, nothing happens when it is 0
int run_scan(pvg_scene* s, uint32_t nv, bool blocks, uint32_t* out, const uint32_t* visit, Timer* tm, bool scratch_ready = false,
             const uint32_t* counts = nullptr /* default: the rectangle counts */, uint32_t rank0 = 0, const uint32_t* only_if = nullptr) {
  cudaStream_t st = s->stream;
  const uint32_t n = nv;
  if (n == 0) return PVG_OK;
  const uint32_t scan_tiles = (n + SCAN_TILE - 1) / SCAN_TILE;
  if (!scratch_ready) {
    TRY(prep_scan(s, st));
    if (tm) tm->cut();
  }
  const bool second = rank0 > 0;
  uint32_t* ticket = reinterpret_cast<uint32_t*>(s->small.as<unsigned char>() + (second ? 96 : 0));
  uint64_t* total = reinterpret_cast<uint64_t*>(s->small.as<unsigned char>() + 8);
  uint64_t* total_out = second ? reinterpret_cast<uint64_t*>(s->small.as<unsigned char>() + 104) : total;
  uint64_t* status = s->scan_status.as<uint64_t>() + (second ? (s->n + SCAN_TILE - 1) / SCAN_TILE : 0);
  if (tm) TRY(tm->begin("scan_counts", PVG_STAGE_DUPLICATE, st));
  if (blocks)
    TRY(launch_chain(tm, scan_counts_kernel<true>, dim3(scan_tiles), dim3(SCAN_THREADS), 0, st, n, s->counts.as<uint32_t>(),
                     s->dkeys[s->visit_side].as<uint64_t>(), visit, out, total_out, status, ticket,
                     s->chunk_owner.as<uint32_t>(), kOwnerChunk, rank0, second ? total : (uint64_t*)nullptr, only_if));
  else
    TRY(launch_chain(tm, scan_counts_kernel<false>, dim3(scan_tiles), dim3(SCAN_THREADS), 0, st, n,
                     counts ? counts : s->counts.as<uint32_t>(), (const uint64_t*)nullptr, visit, out, total,
                     s->scan_status.as<uint64_t>(), ticket, (uint32_t*)nullptr, 0u, 0u, (const uint64_t*)nullptr, (const uint32_t*)nullptr));
  if (tm) TRY(tm->end(st));
  return PVG_OK;
}

// ---- front-first depth order (onesweep.cuh, PVG_OPT_LAZY_DEPTH) ---------------------------------------------------
// dsel (u32 words): the front's histogram region, the back's, two tickets of depth_select_kernel
constexpr size_t kDselWords = 2 * (size_t)DH_WORDS + 4;
inline uint32_t sel_tiles(uint32_t n) { return (n + SEL_TILE - 1) / SEL_TILE; }

// sizes the scratch of a front-first frame and zeroes it on stream zs
int prep_front(pvg_scene* s, cudaStream_t zs) {
  cudaStream_t st = s->stream;
  TRY(s->okeys.reserve((size_t)s->n * 8, st));
  TRY(s->front_idx.reserve((size_t)s->n * 4, st));
  TRY(s->dsel.reserve(kDselWords * 4, st));
  TRY(s->sel_status.reserve((size_t)2 * sel_tiles(s->n) * 8, st));
  CU(cudaMemsetAsync(s->dsel.p, 0, kDselWords * 4, zs));
  CU(cudaMemsetAsync(s->sel_status.p, 0, (size_t)2 * sel_tiles(s->n) * 8, zs));
  return PVG_OK;
}

// cls 0: the pairs below the threshold, to positions [0, F) of buffer pair 1; cls 1: the others, to [F, S) of the pair
// from which the back's passes end in the buffer the front ended in.
int back_out_side(const pvg_scene* s) { return s->visit_side ^ ((3 + s->top_back) & 1); }
int run_depth_select(pvg_scene* s, int cls, const uint32_t* only_if, Timer* tm) {
  cudaStream_t st = s->stream;
  const uint32_t* dh = s->dhist.as<uint32_t>() + s->dhist_side * kDhistWords;
  const FrontCtl* fc = reinterpret_cast<const FrontCtl*>(dh + DH_CTL);
  uint32_t* region = s->dsel.as<uint32_t>() + (size_t)cls * DH_WORDS;
  uint64_t* status = s->sel_status.as<uint64_t>() + (size_t)cls * sel_tiles(s->n);
  uint32_t* ticket = s->dsel.as<uint32_t>() + 2 * (size_t)DH_WORDS + cls;
  const int out_side = cls ? back_out_side(s) : 1;
  uint64_t* lb = s->sort_n.lookback.as<uint64_t>() + (cls ? class_lookback_words(s->n, 0) : 0);
  const uint32_t lb_rows = (uint32_t)class_lookback_rows(s->n, cls), lb_tile = cls ? kDsTile : kDsFrontTile;
  if (tm) TRY(tm->begin("depth_select", PVG_STAGE_DEPTH_SORT, st));
  if (cls)
    TRY(launch_chain(tm, depth_select_kernel<true>, dim3(sel_tiles(s->n)), dim3(SEL_THREADS), 0, st, s->okeys.as<uint64_t>(), s->n, fc,
                     s->dkeys[out_side].as<uint64_t>(), s->dvals[out_side].as<uint32_t>(), (uint32_t*)nullptr, region, status, ticket,
                     (uint32_t)out_side, lb, lb_rows, lb_tile, only_if));
  else
    TRY(launch_chain(tm, depth_select_kernel<false>, dim3(sel_tiles(s->n)), dim3(SEL_THREADS), 0, st, s->okeys.as<uint64_t>(), s->n, fc,
                     s->dkeys[out_side].as<uint64_t>(), s->dvals[out_side].as<uint32_t>(), s->front_idx.as<uint32_t>(), region, status, ticket,
                     (uint32_t)out_side, lb, lb_rows, lb_tile, only_if));
  if (tm) TRY(tm->end(st));
  return PVG_OK;
}

// passes [p0, p1) over one class: small launches whose CTAs loop over tickets (the class's size is in its control block)
// count: an upper bound of the class's pairs known to the host (n before it has read F)
int run_class_passes(pvg_scene* s, int cls, uint32_t count, int p0, int p1, const uint32_t* only_if, Timer* tm) {
  cudaStream_t st = s->stream;
  const uint32_t* region = s->dsel.as<uint32_t>() + (size_t)cls * DH_WORDS;
  const DepthCtl* ctl = reinterpret_cast<const DepthCtl*>(region + DH_CTL);
  const size_t base = cls ? s->front : 0u;
  const size_t tiles = class_lookback_rows(s->n, cls);
  uint64_t* lb = s->sort_n.lookback.as<uint64_t>() + (cls ? class_lookback_words(s->n, 0) : 0);
  uint32_t* tk = s->sort_n.tickets.as<uint32_t>() + cls * DS_PASSES;
  uint64_t* ka = s->dkeys[0].as<uint64_t>() + base; uint32_t* va = s->dvals[0].as<uint32_t>() + base;
  uint64_t* kb = s->dkeys[1].as<uint64_t>() + base; uint32_t* vb = s->dvals[1].as<uint32_t>() + base;
  const unsigned ctas = (unsigned)s->dev.sms * (unsigned)DsCfg::MINB;
  for (int p = 0; p < p0; ++p) lb += tiles * (size_t)(1 << ds_bits(p));
  for (int p = p0; p < p1; ++p) {
    if (tm) TRY(tm->begin("onesweep_pass", PVG_STAGE_DEPTH_SORT, st));
    const uint32_t* hist = region + p * DS_RADIX;
    if (cls == 0) {
      const unsigned fctas = (unsigned)s->dev.sms * (unsigned)DsFrontCfg::MINB;
      if (p < 3) TRY((launch_depth_pass<DS_BITS, false, true, DsFrontCfg>(ka, va, kb, vb, count, p, ctl, hist, lb, tk + p, st, s->dev.ordinal, tm, fctas, only_if)));
      else TRY((launch_depth_pass<DS_TOP_BITS, false, true, DsFrontCfg>(ka, va, kb, vb, count, p, ctl, hist, lb, tk + p, st, s->dev.ordinal, tm, fctas, only_if)));
    } else if (p < 3) TRY((launch_depth_pass<DS_BITS, false, true>(ka, va, kb, vb, count, p, ctl, hist, lb, tk + p, st, s->dev.ordinal, tm, ctas, only_if)));
    else TRY((launch_depth_pass<DS_TOP_BITS, false, true>(ka, va, kb, vb, count, p, ctl, hist, lb, tk + p, st, s->dev.ordinal, tm, ctas, only_if)));
    if (tm) TRY(tm->end(st));
    lb += tiles * (size_t)(1 << ds_bits(p));
  }
  CU(cudaGetLastError());
  return PVG_OK;
}

// The back of a front-first frame: the pairs at and beyond the threshold, selected, ordered behind the front and
// scanned (block entries, continuing the front's offsets). only_if: the parked-tile count (second round) or nullptr.
int run_depth_back(pvg_scene* s, const uint32_t* only_if, Timer* tm) {
  const uint32_t S = (uint32_t)s->survivors, F = s->front;
  if (F >= S) return PVG_OK;
  TRY(run_depth_select(s, 1, only_if, tm));
  TRY(run_class_passes(s, 1, S - F, 0, s->top_back ? 4 : 3, only_if, tm));
  const uint32_t* visit = s->dvals[s->visit_side].as<uint32_t>();
  TRY(run_scan(s, S - F, true, s->boffsets.as<uint32_t>(), visit, tm, true, nullptr, F, only_if));
  return PVG_OK;
}

template <int BITS>
int launch_bin_pass(pvg_scene* s, uint32_t Mb, const uint32_t* bin_start, uint64_t* lookback, uint32_t* ticket) {
  auto kern = bin_pass_kernel<BITS>;
  PVG_ENSURE_SMEM(kern, sizeof(BinPassSmem<BITS>), s->dev.ordinal);
  constexpr uint32_t TILE = BP_THREADS * BP_ITEMS;
  kern<<<(Mb + TILE - 1) / TILE, BP_THREADS, sizeof(BinPassSmem<BITS>), s->stream>>>(
      s->e_bin.as<uint8_t>(), s->e_g.as<uint32_t>(), s->e_mask.as<uint64_t>(), s->s_g.as<uint32_t>(),
      s->s_mask.as<uint64_t>(), Mb, bin_start, lookback, ticket);
  return PVG_OK;
}

template <int BITS>
int launch_bin_emit(pvg_scene* s, uint32_t Mb, const uint32_t* visit, uint32_t blocks_x, const uint32_t* bin_start,
                    uint64_t* lookback, uint32_t* ticket, uint32_t grid, const uint32_t* only_if, uint32_t tile_end) {
  if (s->exact_used) {
    auto kern = bin_emit_kernel<BITS, true>;
    PVG_ENSURE_SMEM(kern, sizeof(BinEmitSmem<BITS>), s->dev.ordinal);
    TRY(launch_chain(&s->timer, kern, dim3(grid), dim3(BP_THREADS), sizeof(BinEmitSmem<BITS>), s->stream,
                     s->nv, Mb, s->boffsets.as<uint32_t>(), s->chunk_owner.as<uint32_t>(), s->dkeys[s->visit_side].as<uint64_t>(), visit,
                     blocks_x, s->s_g.as<uint32_t>(), s->s_mask.as<uint64_t>(), bin_start, lookback, ticket, only_if, s->record.as<float4>(), tile_end));
  } else {
    auto kern = bin_emit_kernel<BITS, false>;
    PVG_ENSURE_SMEM(kern, sizeof(BinEmitSmem<BITS>), s->dev.ordinal);
    TRY(launch_chain(&s->timer, kern, dim3(grid), dim3(BP_THREADS), sizeof(BinEmitSmem<BITS>), s->stream,
                     s->nv, Mb, s->boffsets.as<uint32_t>(), s->chunk_owner.as<uint32_t>(), s->dkeys[s->visit_side].as<uint64_t>(), visit,
                     blocks_x, s->s_g.as<uint32_t>(), s->s_mask.as<uint64_t>(), bin_start, lookback, ticket, only_if, (const float4*)nullptr, tile_end));
  }
  return PVG_OK;
}

// a2 + a3 (instance part) through 8x8-tile block entries (blockbin.cuh): the sorted value list
// lands in vals[0]; ranges come from tile_prefix_kernel.
// Sizes the buffers of the block path from M and Mb and zeroes its tickets and look-back words on stream zs
// (the side stream, while the depth sort is still running on the main one).
// Several regions zeroed by ONE launch: each cudaMemsetAsync is a launch of its own, and four or five of them in a row
// were 12-15 us of stream time whatever their sizes (here 32 B ... 9.6 MB).
struct ZeroList {
  static constexpr int MAX = 6;
  uint32_t* p[MAX];
  uint64_t words[MAX];   // 4-byte words; the regions are 16-byte aligned (256: the allocator's)
  int count;
  void add(void* ptr, size_t bytes) { p[count] = static_cast<uint32_t*>(ptr); words[count] = (bytes + 3) / 4; ++count; }
};
__global__ void __launch_bounds__(256) zero_regions_kernel(const __grid_constant__ ZeroList z) {
  for (int r = 0; r < z.count; ++r) {
    uint4* q = reinterpret_cast<uint4*>(z.p[r]);
    const uint64_t quads = z.words[r] / 4;
    for (uint64_t i = (uint64_t)blockIdx.x * 256 + threadIdx.x; i < quads; i += (uint64_t)gridDim.x * 256) q[i] = make_uint4(0u, 0u, 0u, 0u);
    if (blockIdx.x == 0 && threadIdx.x < (z.words[r] & 3u)) z.p[r][quads * 4 + threadIdx.x] = 0u;
  }
}

int prep_block_bins(pvg_scene* s, const FrameParams& P, cudaStream_t zs) {
  cudaStream_t st = s->stream;
  ZeroList zl = {};
  const uint32_t Mb = (uint32_t)s->Mb;
  const uint32_t nbins = bb_blocks(P.tiles_x) * bb_blocks(P.tiles_y);
  constexpr uint32_t PASS_TILE = BP_THREADS * BP_ITEMS;
  const uint32_t pass_tiles = (Mb + PASS_TILE - 1) / PASS_TILE;
  const uint32_t max_chunks = (Mb + BB_CHUNK - 1) / BB_CHUNK + nbins;
  TRY(s->vals[0].reserve((size_t)s->M * 4, st, 1.125));
  if (!PVG_BIN_FUSED) {
    TRY(s->e_bin.reserve((size_t)Mb + 16, st, 1.125));
    TRY(s->e_g.reserve((size_t)Mb * 4, st, 1.125));
    TRY(s->e_mask.reserve((size_t)Mb * 8, st, 1.125));
  }
  TRY(s->s_g.reserve((size_t)Mb * 4, st, 1.125));
  TRY(s->s_mask.reserve((size_t)Mb * 8, st, 1.125));
  TRY(s->chunk_cnt.reserve((size_t)max_chunks * 64 * 8, st, 1.125));   // look-back words of bin_write
  TRY(s->sort_m.lookback.reserve((size_t)pass_tiles * OS_RADIX * 8, st, 1.25));
  TRY(s->sort_m.tickets.reserve((size_t)OS_MAX_PASSES * 4, st));
  TRY(s->chunk_owner.reserve(((size_t)Mb / kOwnerChunk + 2) * 4, st, 1.125));
  zl.add(s->sort_m.tickets.p, 32);   // emit, write (round 0), write (round 1), write (completion), exact count
  if (s->exact_used) {
    const size_t tiles = (size_t)P.tiles_x * P.tiles_y;
    TRY(s->tile_count.reserve(tiles * 4, st));
    TRY(s->counts_exact.reserve((size_t)s->n * 4, st));
    zl.add(s->tile_count.p, tiles * 4);
    zl.add(s->counts_exact.p, (size_t)s->n * 4);
  }
  zl.add(s->chunk_cnt.p, (size_t)max_chunks * 64 * 8);
  if (s->lazy_chunks > 0 && !s->exact_used) {
    const size_t tiles = (size_t)P.tiles_x * P.tiles_y;
    TRY(s->unf.reserve(kUnfHead + tiles * 8, st));
    TRY(s->lazy_state.reserve((size_t)5 * P.width * P.height * 4, st));
    zl.add(s->unf.p, kUnfHead + tiles * 4);   // masks, count and lim; the list is written before it is read
  }
  zl.add(s->sort_m.lookback.p, (size_t)pass_tiles * OS_RADIX * 8);
  Timer& tm = s->timer;
  tm.cut();
  TRY(tm.begin("zero_scratch", PVG_STAGE_SORT, zs));
  zero_regions_kernel<<<std::max(1, s->dev.sms * 4), 256, 0, zs>>>(zl);
  TRY(tm.end(zs));
  tm.cut();
  CU(cudaGetLastError());
  return PVG_OK;
}

#if PVG_BIN_FUSED
// bin_emit over the next `grid` tiles of 4096 entries (the ticket goes on counting across launches)
// loop: the CTAs of the launch loop over tickets up to the last tile (a grid of at most two CTAs per SM)
int run_bin_emit(pvg_scene* s, const FrameParams& P, const uint32_t* visit, uint32_t grid, const uint32_t* only_if, bool loop = false) {
  const uint32_t tile_end = loop ? s->emit_tiles : 0u;
  if (loop) grid = std::min(grid, (uint32_t)s->dev.sms * (uint32_t)PVG_BP_MINB);
  const uint32_t blocks_x = bb_blocks(P.tiles_x), nbins = blocks_x * bb_blocks(P.tiles_y);
  uint32_t* bin_start = s->bin_tables.as<uint32_t>();
  uint32_t* ticket = s->sort_m.tickets.as<uint32_t>();
  int rc = PVG_ERR_BAD_OPTION;
  switch (std::max(1, ceil_log2(nbins))) {
#define PVG_CASE(B) case B: rc = launch_bin_emit<B>(s, (uint32_t)s->Mb, visit, blocks_x, bin_start, s->sort_m.lookback.as<uint64_t>(), ticket, grid, only_if, tile_end); break;
    PVG_CASE(1) PVG_CASE(2) PVG_CASE(3) PVG_CASE(4) PVG_CASE(5) PVG_CASE(6) PVG_CASE(7) PVG_CASE(8)
#undef PVG_CASE
    default: break;
  }
  return rc;
}
#endif

// shade_kernel over the depth ranks (r_lo, r_hi] given by device words (nullptr: from the start / to the last survivor)
int run_shade(pvg_scene* s, const FrameParams& P, const uint32_t* r_lo, const uint32_t* r_hi, const uint32_t* only_if,
              cudaStream_t on = nullptr) {
  const Model* m = s->model;
  if (s->nv == 0) return PVG_OK;
  shade_kernel<<<(s->nv + 255) / 256, 256, 0, on ? on : s->stream>>>(P, s->n, s->nv, s->visit_last, r_lo, r_hi, only_if,
                                                                      m->A0.as<float4>(), m->A1.as<float4>(), m->A2.as<float4>(),
                                                                      m->A3.as<float4>(), m->SH.as<float4>(), s->record.as<float4>(),
                                                                      s->featw_last);
  return PVG_OK;
}

// every Gaussian's record, in index order (zeros for the culled ones)
int run_shade_all(pvg_scene* s, const FrameParams& P, const uint32_t* only_if, cudaStream_t on = nullptr) {
  const Model* m = s->model;
  cudaStream_t st = on ? on : s->stream;
  const unsigned grid = std::min<unsigned>((s->n + 255) / 256, (unsigned)s->dev.sms * 8u);
  return launch_chain(&s->timer, shade_all_kernel, dim3(grid), dim3(256), 0, st, P, s->n, s->counts.as<uint32_t>(),
                      only_if, m->A0.as<float4>(), m->A1.as<float4>(), m->A2.as<float4>(), m->A3.as<float4>(), m->SH.as<float4>(),
                      s->record.as<float4>(), s->featw_last);
}

// bin_write over the chunks kin_lo <= kin < kin_hi of every block; only_unfinished: the tiles the first blend
// phase marked. ticket_slot: which zeroed ticket of sort_m.tickets this launch consumes.
int launch_bin_write(pvg_scene* s, const FrameParams& P, uint32_t kin_lo, uint32_t kin_hi, bool only_unfinished, int ticket_slot) {
  const uint32_t Mb = (uint32_t)s->Mb;
  const uint32_t blocks_x = bb_blocks(P.tiles_x), nbins = blocks_x * bb_blocks(P.tiles_y);
  const uint32_t max_chunks = (Mb + BB_CHUNK - 1) / BB_CHUNK + nbins;
  uint32_t* bin_start = s->bin_tables.as<uint32_t>();   // written by tile_prefix_kernel
  const uint32_t launch_chunks = (kin_lo == 0 && kin_hi < (1u << 30)) ? std::min<uint64_t>((uint64_t)nbins * kin_hi, 0x7FFFFFFFull) : max_chunks;
  unsigned grid = (launch_chunks + BW_CHUNKS_PER_CTA - 1) / BW_CHUNKS_PER_CTA;
  // the second round (parked tiles only) usually finds nothing to do: a grid of four CTAs per SM that loops over tickets
  const uint32_t loop = only_unfinished ? 1u : 0u;
  if (loop) grid = std::min(grid, (unsigned)s->dev.sms * 4u);
  return launch_chain(&s->timer, bin_write_kernel, dim3(grid), dim3(BW_THREADS), 0, s->stream,
      s->s_g.as<uint32_t>(), s->s_mask.as<uint64_t>(), bin_start, bin_start + 257, s->ranges.as<uint2>(), (uint32_t)P.tiles_x,
      (uint32_t)P.tiles_y, blocks_x, s->chunk_cnt.as<uint64_t>(), s->sort_m.tickets.as<uint32_t>() + ticket_slot,
      s->vals[0].as<uint32_t>(), kin_lo, kin_hi, only_unfinished ? s->unf.as<unsigned long long>() : (unsigned long long*)nullptr,
      reinterpret_cast<const uint32_t*>(s->unf.as<unsigned char>() + 2048),
      (kin_lo == 0 && kin_hi < (1u << 30)) ? reinterpret_cast<uint32_t*>(s->unf.as<unsigned char>() + kUnfHead) : (uint32_t*)nullptr,
      (s->lazy_used && s->emit_first && s->emit_first < s->emit_tiles)
          ? s->sort_m.lookback.as<uint64_t>() + (size_t)(s->emit_first - 1) * s->emit_radix : (uint64_t*)nullptr, loop);
}

// a2 + a3 (instance part) through 8x8-tile block entries (blockbin.cuh), after prep_block_bins: the sorted value
// list lands in vals[0]; ranges come from tile_prefix_kernel.
int run_block_bins(pvg_scene* s, const FrameParams& P, const uint32_t* visit, Timer* tm) {
  cudaStream_t st = s->stream;
  const uint32_t Mb = (uint32_t)s->Mb;
  const uint32_t blocks_x = bb_blocks(P.tiles_x), nbins = blocks_x * bb_blocks(P.tiles_y);
  const int bits = std::max(1, ceil_log2(nbins));
#if !PVG_BIN_FUSED
  uint32_t* bin_start = s->bin_tables.as<uint32_t>();   // written by tile_prefix_kernel
  uint32_t* ticket = s->sort_m.tickets.as<uint32_t>();
  int rc = PVG_ERR_BAD_OPTION;
#endif
#if PVG_BIN_FUSED
  // lazy lists: only the first slab of the entries (in depth order) is formed now; render_impl emits the rest if
  // the first blend phase parks a tile
  s->lazy_used = s->lazy_chunks > 0 && !s->exact_used;   // exact lists are counted: every entry is formed and refined
  const uint32_t emit_tiles = (Mb + BF_TILE - 1) / BF_TILE;
  s->emit_first = s->lazy_used ? lazy_emit_first(Mb, s->lazy_slab, P.lazy_min_tiles) : emit_tiles;
  s->emit_tiles = emit_tiles;
  s->emit_radix = 1u << bits;
  s->visit_last = visit;
  if (s->light && !s->front_used) {
    // the records of the Gaussians that own the first slab's entries (depth ranks 0 .. owner of the slab's end), on
    // the side stream: a latency-bound gather that overlaps the equally latency-bound bin_emit and bin_write
    cudaStream_t sd = s->side;
    CU(cudaEventRecord(s->ev_fork, st));
    CU(cudaStreamWaitEvent(sd, s->ev_fork, 0));
    tm->cut();
    TRY(tm->begin("shade", PVG_STAGE_PREPROCESS, sd));
    TRY(run_shade(s, P, nullptr, s->emit_first < s->emit_tiles ? s->chunk_owner.as<uint32_t>() + s->emit_first : nullptr, nullptr, sd));
    TRY(tm->end(sd));
    CU(cudaEventRecord(s->ev_join, sd));
  }
  TRY(tm->begin("bin_emit", PVG_STAGE_SORT, st));
  TRY(run_bin_emit(s, P, visit, s->emit_first, nullptr));
  TRY(tm->end(st));
  if (s->exact_used) {
    // exact lists: the masks are refined, so the tile counts are counted (not taken from the rectangles) and the
    // ranges rebuilt from them before the lists are written
    const uint32_t nb = blocks_x * bb_blocks(P.tiles_y);
    const uint32_t max_chunks = (Mb + BB_CHUNK - 1) / BB_CHUNK + nb;
    uint32_t* bin_start = s->bin_tables.as<uint32_t>();
    TRY(tm->begin("exact_count", PVG_STAGE_RANGES, st));
    exact_count_kernel<<<(max_chunks + BW_CHUNKS_PER_CTA - 1) / BW_CHUNKS_PER_CTA, BW_THREADS, 0, st>>>(
        s->s_g.as<uint32_t>(), s->s_mask.as<uint64_t>(), bin_start, bin_start + 257, (uint32_t)P.tiles_x, (uint32_t)P.tiles_y,
        blocks_x, s->sort_m.tickets.as<uint32_t>() + 4, s->tile_count.as<uint32_t>(), s->counts_exact.as<uint32_t>());
    TRY(tm->end(st));
    TRY(tm->begin("exact_ranges", PVG_STAGE_RANGES, st));
    exact_ranges_kernel<<<1, 1024, 0, st>>>(s->tile_count.as<uint32_t>(), (uint32_t)P.tiles_x * (uint32_t)P.tiles_y,
                                            s->ranges.as<uint2>(), reinterpret_cast<uint64_t*>(s->small.as<unsigned char>() + 40),
                                            s->d_total);
    TRY(tm->end(st));
  }
#else
  TRY(tm->begin("bin_expand", PVG_STAGE_DUPLICATE, st));
  bin_expand_kernel<<<(Mb + BE_CHUNK - 1) / BE_CHUNK, BE_THREADS, 0, st>>>(
      s->nv, Mb, s->boffsets.as<uint32_t>(), s->chunk_owner.as<uint32_t>(), s->dkeys[s->visit_side].as<uint64_t>(), visit, blocks_x,
      s->e_bin.as<uint8_t>(),
      s->e_g.as<uint32_t>(), s->e_mask.as<uint64_t>());
  TRY(tm->end(st));

  TRY(tm->begin("bin_pass", PVG_STAGE_SORT, st));
  switch (bits) {
#define PVG_CASE(B) case B: rc = launch_bin_pass<B>(s, Mb, bin_start, s->sort_m.lookback.as<uint64_t>(), ticket); break;
    PVG_CASE(1) PVG_CASE(2) PVG_CASE(3) PVG_CASE(4) PVG_CASE(5) PVG_CASE(6) PVG_CASE(7) PVG_CASE(8)
#undef PVG_CASE
    default: break;
  }
  TRY(rc);
  TRY(tm->end(st));
#endif

  // the tile lists: all of them, or (lazy) only as far as the first lazy_chunks chunks of every block reach --
  // render_impl runs the second round after the first blend phase
#if !PVG_BIN_FUSED
  s->lazy_used = s->lazy_chunks > 0 && !s->exact_used;
  s->emit_first = s->emit_tiles = 0;
#endif
  s->lists_complete = !s->lazy_used;
  s->visit_last = visit;
  if (s->front_used) {   // the ranges (tile_prefix_kernel, tile level): bin_write is their first reader
    CU(cudaStreamWaitEvent(st, s->ev_join, 0));
    tm->cut();
  }
  TRY(tm->begin("bin_write", PVG_STAGE_SORT, st));
  TRY(launch_bin_write(s, P, 0u, s->lazy_used ? (uint32_t)s->lazy_chunks : 0xFFFFFFFFu, false, 1));
  TRY(tm->end(st));
  if (s->light && !s->front_used) {   // the blend reads the records
    CU(cudaStreamWaitEvent(st, s->ev_join, 0));
    tm->cut();
  }
  // (front-first frames: shade_list_kernel ran on the aux stream ahead of the zeroing kernel whose event, ev_zero, the
  // main stream waited for before bin_emit -- nothing sits between bin_write and the blend, which is launched as its
  // programmatic dependent)
  CU(cudaGetLastError());
  s->sorted_side = 0;
  return PVG_OK;
}

// PVG_R2_TAIL=1: the second round of the lazy lists is launched from the device, by a one-thread gate kernel after the
// first blend phase, only if a tile parked (round2.cu); 0: the host launches it every frame and each kernel looks at
// the parked count.
#ifndef PVG_R2_TAIL
#define PVG_R2_TAIL 1
#endif

#ifndef PVG_FRONT_FUSED
#define PVG_FRONT_FUSED 1
#endif
extern "C" int pvg_r2_gate(int device, void* stream, const void* params, const void* chain, const void* lazy, int which,
                           const void* ranges, const void* vals, const void* record, float* out_rgb, float* out_depth,
                           float* out_alpha, unsigned long long* counters, const float* featw, int pdl);

// The launches of the second round, described for r2_tail_launch: the same kernels, grids and arguments as the host
// path further down (run_depth_back, run_shade_all, run_bin_emit, launch_bin_write, the second blend phase).
int fill_r2(pvg_scene* s, const FrameParams& P, uint32_t band_tiles, R2Chain* out) {
  R2Chain c = {};
  const uint32_t S = (uint32_t)s->survivors, F = s->front, n = s->n;
  const uint32_t sms = (uint32_t)s->dev.sms;
  const bool more = s->emit_first < s->emit_tiles;
  c.enabled = 1;
  c.n = n;
  c.counts = s->counts.as<uint32_t>();
  c.visit = s->dvals[s->visit_side].as<uint32_t>();
  c.scan_keys = s->dkeys[s->visit_side].as<uint64_t>();
  c.boffsets = s->boffsets.as<uint32_t>();
  c.chunk_owner = s->chunk_owner.as<uint32_t>();
  c.back = (more && s->front_used && F < S) ? 1u : 0u;
  if (c.back) {
    const int side = back_out_side(s);
    c.okeys = s->okeys.as<uint64_t>();
    c.fc = reinterpret_cast<const FrontCtl*>(s->dhist.as<uint32_t>() + s->dhist_side * kDhistWords + DH_CTL);
    c.sel_keys = s->dkeys[side].as<uint64_t>(); c.sel_vals = s->dvals[side].as<uint32_t>();
    c.sel_region = s->dsel.as<uint32_t>() + DH_WORDS;
    c.sel_status = s->sel_status.as<uint64_t>() + sel_tiles(n);
    c.sel_ticket = s->dsel.as<uint32_t>() + 2 * (size_t)DH_WORDS + 1;
    c.sel_side = (uint32_t)side; c.sel_grid = sel_tiles(n);
    c.lb = s->sort_n.lookback.as<uint64_t>() + class_lookback_words(n, 0);
    c.lb_rows = (uint32_t)class_lookback_rows(n, 1); c.lb_tile = kDsTile;
    c.ka = s->dkeys[0].as<uint64_t>() + F; c.va = s->dvals[0].as<uint32_t>() + F;
    c.kb = s->dkeys[1].as<uint64_t>() + F; c.vb = s->dvals[1].as<uint32_t>() + F;
    c.back_count = S - F; c.passes = s->top_back ? 4u : 3u;
    c.pass_grid = std::max(1u, std::min((S - F + kDsTile - 1) / kDsTile, sms * (uint32_t)DsCfg::MINB));
    c.pass_tickets = s->sort_n.tickets.as<uint32_t>() + DS_PASSES;
    c.scan_grid = (S - F + SCAN_TILE - 1) / SCAN_TILE;
    c.scan_total = reinterpret_cast<uint64_t*>(s->small.as<unsigned char>() + 104);
    c.scan_init = reinterpret_cast<const uint64_t*>(s->small.as<unsigned char>() + 8);
    c.scan_status = s->scan_status.as<uint64_t>() + (n + SCAN_TILE - 1) / SCAN_TILE;
    c.scan_ticket = reinterpret_cast<uint32_t*>(s->small.as<unsigned char>() + 96);
    c.owner_chunk = kOwnerChunk; c.rank0 = F;
  }
  const Model* m = s->model;
  c.shade = (more && s->light) ? 1u : 0u;
  c.shade_grid = std::min<uint32_t>((n + 255) / 256, sms * 8u);
  c.A0 = m->A0.as<float4>(); c.A1 = m->A1.as<float4>(); c.A2 = m->A2.as<float4>(); c.A3 = m->A3.as<float4>(); c.SH = m->SH.as<float4>();
  c.record = s->record.as<float4>(); c.featw = s->featw_last;
  const uint32_t blocks_x = bb_blocks(P.tiles_x), nbins = blocks_x * bb_blocks(P.tiles_y);
  const uint32_t Mb = (uint32_t)s->Mb;
  c.emit = more ? 1u : 0u;
  c.emit_grid = std::max(1u, std::min(s->emit_tiles - std::min(s->emit_tiles, s->emit_first), sms * (uint32_t)PVG_BP_MINB));
  c.emit_bits = (uint32_t)std::max(1, ceil_log2(nbins));
  c.nv = c.back ? S : s->nv; c.Mb = Mb; c.blocks_x = blocks_x; c.emit_tiles = s->emit_tiles;
  c.s_g = s->s_g.as<uint32_t>(); c.s_mask = s->s_mask.as<uint64_t>(); c.bin_start = s->bin_tables.as<uint32_t>();
  c.emit_lookback = s->sort_m.lookback.as<uint64_t>(); c.emit_ticket = s->sort_m.tickets.as<uint32_t>();
  const uint32_t max_chunks = (Mb + BB_CHUNK - 1) / BB_CHUNK + nbins;
  c.write_grid = std::max(1u, std::min((max_chunks + BW_CHUNKS_PER_CTA - 1) / BW_CHUNKS_PER_CTA, sms * 4u));
  c.ranges = s->ranges.as<uint2>(); c.tiles_x = (uint32_t)P.tiles_x; c.tiles_y = (uint32_t)P.tiles_y;
  c.chunk_cnt = s->chunk_cnt.as<uint64_t>(); c.write_ticket = s->sort_m.tickets.as<uint32_t>() + 2;
  c.vals = s->vals[0].as<uint32_t>(); c.kin_lo = (uint32_t)s->lazy_chunks;
  c.want_mask = s->unf.as<unsigned long long>();
  c.want_count = reinterpret_cast<const uint32_t*>(s->unf.as<unsigned char>() + 2048);
  c.avail = (s->lazy_used && s->emit_first && s->emit_first < s->emit_tiles)
                ? s->sort_m.lookback.as<uint64_t>() + (size_t)(s->emit_first - 1) * s->emit_radix : (const uint64_t*)nullptr;
  c.blend_grid = std::max(1u, std::min(band_tiles, sms * 8u));
  *out = c;
  return PVG_OK;
}

int render_impl(pvg_scene* s, const pvg_camera* cam, const pvg_state* state, float* out_rgb, float* out_depth,
                float* out_alpha) {
  FrameParams P;
  TRY(fill_frame(s, cam, state, &P));
  DeviceGuard guard(s->dev.ordinal);
  cudaStream_t st = s->stream;
  Timer& tm = s->timer;
  tm.cut();
  s->presort_used = s->presort; s->keep_unsorted_used = s->keep_unsorted; s->lazy_chunks_used = s->lazy_chunks;
  tm.next_frame();
  if (!tm.accumulate) { if (tm.frame_on) tm.reset(); } else tm.cut();
  const uint32_t n = s->n;
  const uint32_t tiles = (uint32_t)P.tiles_x * (uint32_t)P.tiles_y;
  s->tiles_x = P.tiles_x; s->tiles_y = P.tiles_y;
  s->rendered = false;
  s->visit_tail_done = false;
  TRY(s->ranges.reserve((size_t)tiles * 8, st));

  const int tile_bits = std::max(1, ceil_log2(tiles));
  s->sort_begin = s->presort ? 32 : 0;
  s->sort_end = 32 + tile_bits;

  // which list builder (blockbin.cuh needs the depth order, <= 256 blocks and 8-bit tile coordinates)
  const uint32_t blocks_x = bb_blocks(P.tiles_x), blocks_y = bb_blocks(P.tiles_y);
  const bool block = s->presort && s->block && P.pack_rect && blocks_x * blocks_y <= (uint32_t)BB_MAX_BINS;
  s->block_used = block;
  s->last_P = P;

  // lazy lists: the records (conic, colour: 48 B written, 192 B of SH read per survivor) are left to shade_kernel,
  // which forms them for the Gaussians in front only -- unless a tile parks; and only that front is ordered
  s->exact_used = block && s->exact_tiles && PVG_BIN_FUSED;
  s->light = block && s->lazy_chunks > 0 && PVG_BIN_FUSED && !s->exact_used;
  s->front_used = s->light && (s->lazy_depth >= 2 || (s->lazy_depth == 1 && n >= PVG_LAZY_DEPTH_MIN_N));
  s->depth_complete = !s->front_used;
  s->records_complete = !s->light;

  // scratch of the depth sort and of the scan: sized by n, zeroed on the side stream while preprocess runs
  if (s->presort) {
    cudaStream_t sd = s->side;
    CU(cudaStreamWaitEvent(st, s->ev_zero, 0));   // normally long past; matters only after a frame that stopped early
    CU(cudaEventRecord(s->ev_start, st));
    CU(cudaStreamWaitEvent(sd, s->ev_start, 0));
    TRY(prep_depth_sort(n, st, sd, s->sort_n, s->front_used));
    if (s->front_used) TRY(prep_front(s, sd));
    // the depth histogram is accumulated by preprocess into one half of dhist; the other half is zeroed here for
    // the next frame (its last readers, the previous frame's passes, are behind ev_start)
    s->dhist_side ^= 1;
    CU(cudaMemsetAsync(s->dhist.as<uint32_t>() + (s->dhist_side ^ 1) * kDhistWords, 0, kDhistWords * 4, sd));
    TRY(prep_scan(s, sd));
    CU(cudaEventRecord(s->ev_zero, sd));
  }

  // a1 preprocess
  uint64_t* dk = s->presort ? (s->front_used ? s->okeys.as<uint64_t>() : s->dkeys[0].as<uint64_t>()) : nullptr;
  uint32_t* dv = s->presort ? s->dvals[0].as<uint32_t>() : nullptr;
  float* featw = nullptr;
  if (P.target == 1) {
    TRY(s->featw.reserve((size_t)n * 4, st));
    featw = s->featw.as<float>();
  }
  s->featw_last = featw;
  TRY(tm.begin("preprocess", PVG_STAGE_PREPROCESS, st));
  {
    const unsigned pgrid = (n + 256 * PRE_CHUNKS - 1) / (256 * PRE_CHUNKS);
    uint32_t* dh = s->presort ? s->dhist.as<uint32_t>() + s->dhist_side * kDhistWords : nullptr;
    const Model* m = s->model;
    if (s->front_used)
      preprocess_kernel<PRE_GEO, true><<<pgrid, 256, 0, st>>>(P, n, m->shflag.as<uint8_t>(), m->A0.as<float4>(), m->A1.as<float4>(),
                                                          m->A2.as<float4>(), m->A3.as<float4>(), m->SH.as<float4>(),
                                                          s->record.as<float4>(), s->tileinfo.as<uint4>(),
                                                          s->counts.as<uint32_t>(), dk, dv, featw, dh, s->d_total);
    else if (s->light)
      preprocess_kernel<PRE_GEO, false><<<pgrid, 256, 0, st>>>(P, n, m->shflag.as<uint8_t>(), m->A0.as<float4>(), m->A1.as<float4>(),
                                                          m->A2.as<float4>(), m->A3.as<float4>(), m->SH.as<float4>(),
                                                          s->record.as<float4>(), s->tileinfo.as<uint4>(),
                                                          s->counts.as<uint32_t>(), dk, dv, featw, dh, s->d_total);
    else
      preprocess_kernel<PRE_ALL, false><<<pgrid, 256, 0, st>>>(P, n, m->shflag.as<uint8_t>(), m->A0.as<float4>(), m->A1.as<float4>(),
                                                          m->A2.as<float4>(), m->A3.as<float4>(), m->SH.as<float4>(),
                                                          s->record.as<float4>(), s->tileinfo.as<uint4>(),
                                                          s->counts.as<uint32_t>(), dk, dv, featw, dh, s->d_total);
  }
  TRY(tm.end(st));
  if (s->front_used) {
    CU(cudaEventRecord(s->ev_pre, st));   // the host waits for preprocess alone: its last CTA hands over M, Mb, S and F
    tm.cut();
  }

  const uint32_t* visit = nullptr;
  s->visit_side = 0;
  uint64_t M = 0;
  s->Mb = 0;
  if (s->presort) {
    // a4 + the histograms of a3 + the block tables, from the rectangles alone (no pass over the
    // instances), on the side stream: they overlap the depth sort, and the host reads M and Mb
    // (they size the frame's buffers) while the depth sort is still running
    cudaStream_t sd = s->side;
    CU(cudaStreamWaitEvent(st, s->ev_zero, 0));
    constexpr size_t kMaxDyn = 200 * 1024;
    PVG_ENSURE_SMEM(tile_prefix_kernel, kMaxDyn, s->dev.ordinal);
    PVG_ENSURE_SMEM(tile_grid_kernel, kMaxDyn, s->dev.ordinal);
    const size_t grid_bytes = ((size_t)tilegrid_cells(P.tiles_x, P.tiles_y) +
                               (block ? (size_t)tilegrid_cells((int)blocks_x, (int)blocks_y) : 0)) * 4;   // + 1 cell: survivor count
    const int use_smem = grid_bytes <= kMaxDyn ? 1 : 0;
    TRY(s->tilegrid.reserve(grid_bytes + 4, st));
    TRY(s->sort_m.hist.reserve((size_t)OS_MAX_PASSES * OS_RADIX * 4, st));
    TRY(s->bin_tables.reserve(4096, st));   // bin_start[257] | chunk_start[257]
    int* grid = s->tilegrid.as<int>();
    CU(cudaMemsetAsync(grid, 0, grid_bytes + 4, sd));   // beside preprocess: the side stream waits for it only now
    CU(cudaEventRecord(s->ev_fork, st));
    CU(cudaStreamWaitEvent(sd, s->ev_fork, 0));
    tm.cut();
    TRY(tm.begin("tile_grid", PVG_STAGE_RANGES, sd));
    tile_grid_kernel<<<std::min<unsigned>((n + TG_THREADS - 1) / TG_THREADS, (unsigned)s->dev.sms), TG_THREADS,
                       use_smem ? grid_bytes : 0, sd>>>(s->tileinfo.as<uint4>(), n, P.tiles_x, P.tiles_y, use_smem,
                                                        block ? 1 : 0, grid);
    TRY(tm.end(sd));
    uint64_t* totals = reinterpret_cast<uint64_t*>(s->small.as<unsigned char>() + 16);
    // front-first frames: the block level first, in a launch of its own -- it is all bin_emit waits for
    for (int parts : {s->front_used ? 2 : 3, s->front_used ? 1 : 0}) {
      if (!parts) break;
      TRY(tm.begin(parts == 2 ? "block_prefix" : "tile_prefix", PVG_STAGE_RANGES, sd));
      tile_prefix_kernel<<<1, TB_THREADS, use_smem ? grid_bytes : 0, sd>>>(
          grid, P.tiles_x, P.tiles_y, use_smem, block ? 1 : 0, parts, make_sort_plan(s->sort_begin, s->sort_end),
          s->ranges.as<uint2>(), s->sort_m.hist.as<uint32_t>(), totals, s->bin_tables.as<uint32_t>(),
          s->bin_tables.as<uint32_t>() + 257, s->d_total);
      TRY(tm.end(sd));
      if (parts == 2) CU(cudaEventRecord(s->ev_blocks, sd));
    }
    CU(cudaEventRecord(s->ev_join, sd));
    tm.cut();

    if (s->front_used) {
      // a3 (n-key part), front first: the pairs below preprocess's threshold are compacted and ordered -- launched
      // before the host wait (launches that loop over tickets: the front's size is still on the device)
      TRY(run_depth_select(s, 0, nullptr, &tm));
      {
        // the records of the front, from the compacted list (they do not depend on the order), on a stream of their own
        cudaStream_t ax = s->aux;
        const Model* m = s->model;
        const FrontCtl* fc = reinterpret_cast<const FrontCtl*>(s->dhist.as<uint32_t>() + s->dhist_side * kDhistWords + DH_CTL);
        CU(cudaEventRecord(s->ev_sel, st));
        CU(cudaStreamWaitEvent(ax, s->ev_sel, 0));
        tm.cut();
        TRY(tm.begin("shade", PVG_STAGE_PREPROCESS, ax));
        shade_list_kernel<<<std::min<unsigned>((n + 255) / 256, (unsigned)s->dev.sms * 8u), 256, 0, ax>>>(
            P, n, &fc->front, s->front_idx.as<uint32_t>(), m->A0.as<float4>(), m->A1.as<float4>(), m->A2.as<float4>(),
            m->A3.as<float4>(), m->SH.as<float4>(), s->record.as<float4>(), featw);
        TRY(tm.end(ax));
        CU(cudaEventRecord(s->ev_aux, ax));
      }
      // PVG_FRONT_FUSED=1: the front's passes and scan are launched after the host wait, when its size is known -- as
      // one grid when its tiles fit the GPU at once (front_sort.cuh); the selection covers the host's latency.
      // 0: the passes are launched here, before the wait, as launches that loop over tickets.
      if (!PVG_FRONT_FUSED) TRY(run_class_passes(s, 0, n, 0, 3, nullptr, &tm));
      CU(cudaEventSynchronize(s->ev_pre));
      s->prev_parked = s->h_total[3];   // the frame before has completed (same stream): its parked count
      M = s->h_total[0];
      s->Mb = s->h_total[1];
      s->survivors = s->h_total[4];
      s->front = (uint32_t)s->h_total[8];
      s->top_front = (int)(s->h_total[9] & 1u);
      s->top_back = (int)((s->h_total[9] >> 1) & 1u);
      s->nv = s->front;
      s->visit_side = s->top_front ? 1 : 0;
      visit = s->dvals[s->visit_side].as<uint32_t>();
      const uint32_t ftiles = (s->front + kDsFrontTile - 1) / kDsFrontTile;
      const bool fused = PVG_FRONT_FUSED && s->dev.coop && s->front > 0 && ftiles <= (uint32_t)s->dev.sms * 2u;
      if (PVG_FRONT_FUSED && !fused) TRY(run_class_passes(s, 0, s->front, 0, 3, nullptr, &tm));
      if (!fused && s->top_front) TRY(run_class_passes(s, 0, s->front, 3, 4, nullptr, &tm));
      if (M >= (1ull << 32) - 65536 || s->Mb >= (1ull << 32) - 65536) return PVG_ERR_INSTANCE_OVERFLOW;
      s->M = M;
      if (M > 0) {
        // the block path's scratch, sized here and zeroed on the aux stream behind shade_list_kernel, beside the sort
        // (on the main stream the five memsets -- 14 MB -- sat between the sort and bin_emit: 15 us of the critical
        // path. On a stream of their own they run beside the selection instead, and the frame got 14-16 us SLOWER: a CTA
        // of depth_select_kernel takes a whole SM's registers and has to wait for whatever got onto the SMs first.)
        TRY(prep_block_bins(s, P, s->aux));
        CU(cudaEventRecord(s->ev_zero, s->aux));
      }
      if (fused) {
        static_assert(kDsFrontTile == (uint32_t)FSORT_TILE, "front_sort_kernel runs the front's tile shape");
        using Smem = OnesweepSmem<FSORT_THREADS, FSORT_ITEMS, DS_BITS>;
        PVG_ENSURE_SMEM(front_sort_kernel, sizeof(Smem), s->dev.ordinal);
        uint32_t* region = s->dsel.as<uint32_t>();
        TRY(tm.begin("front_sort_scan", PVG_STAGE_DEPTH_SORT, st));
        {
          // a COOPERATIVE launch: the grid waits on itself (grid_barrier), so all of its CTAs must be resident together
          // whatever else shares the device -- a second frame in flight (pvg_fork_scene) runs the same kernel, and two
          // such grids admitted half each would wait for one another for ever. The attribute makes the co-residency the
          // driver's guarantee instead of an assumption (no programmatic dependent launch for this kernel then).
          cudaLaunchConfig_t cfg = {};
          cfg.gridDim = dim3(ftiles); cfg.blockDim = dim3(FSORT_THREADS); cfg.dynamicSmemBytes = sizeof(Smem); cfg.stream = st;
          cudaLaunchAttribute at[1];
          at[0].id = cudaLaunchAttributeCooperative;
          at[0].val.cooperative = 1;
          cfg.attrs = at; cfg.numAttrs = 1;
          const cudaError_t launched = (cudaLaunchKernelEx(&cfg, front_sort_kernel, s->dkeys[0].as<uint64_t>(), s->dvals[0].as<uint32_t>(),
                                s->dkeys[1].as<uint64_t>(), s->dvals[1].as<uint32_t>(), (const uint32_t*)region,
                                s->sort_n.lookback.as<uint64_t>(), (uint32_t)class_lookback_rows(s->n, 0),
                                s->sort_n.tickets.as<uint32_t>(), s->sort_n.tickets.as<uint32_t>() + 2 * DS_PASSES,
                                s->boffsets.as<uint32_t>(), reinterpret_cast<uint64_t*>(s->small.as<unsigned char>() + 8),
                                s->scan_status.as<uint64_t>(), s->small.as<uint32_t>(),
                                M > 0 ? s->chunk_owner.as<uint32_t>() : (uint32_t*)nullptr, (uint32_t)kOwnerChunk));
          CU(launched);
          tm.pdl_open = true; tm.pdl_stream = st;   // the next kernel of the chain may still be ITS programmatic dependent
        }
        TRY(tm.end(st));
      } else {
        TRY(run_scan(s, s->nv, true, s->boffsets.as<uint32_t>(), visit, &tm, true));
      }
      CU(cudaStreamWaitEvent(st, s->ev_blocks, 0));   // bin_start, chunk_start (tile_prefix_kernel, block level); run_block_bins waits for the ranges
      tm.cut();
    } else {
    // a3 (n-key part): depth order of the survivors
    TRY(run_depth_sort(s->dev, n, s->dkeys[0].as<uint64_t>(), s->dvals[0].as<uint32_t>(), s->dkeys[1].as<uint64_t>(),
                       s->dvals[1].as<uint32_t>(), s->dhist.as<uint32_t>() + s->dhist_side * kDhistWords, st, s->sort_n, &tm, 0, 3));

    // the one host wait of the frame, hidden behind the depth sort: the totals of the tile grid, and what preprocess's
    // last CTA decided for the depth sort (S, and which buffer the sorted pairs end in)
    CU(cudaEventSynchronize(s->ev_join));
    CU(cudaStreamWaitEvent(st, s->ev_join, 0));
    tm.cut();
    s->prev_parked = s->h_total[3];
    M = s->h_total[0];
    s->Mb = block ? s->h_total[1] : 0;
    s->survivors = s->h_total[4];
    s->nv = (uint32_t)s->h_total[4];
    s->visit_side = (int)s->h_total[5];
    visit = s->dvals[s->visit_side].as<uint32_t>();
    if (!(s->h_total[6] & 8u))   // the top digit is not constant: its pass is needed
      TRY(run_depth_sort(s->dev, n, s->dkeys[0].as<uint64_t>(), s->dvals[0].as<uint32_t>(), s->dkeys[1].as<uint64_t>(),
                         s->dvals[1].as<uint32_t>(), s->dhist.as<uint32_t>() + s->dhist_side * kDhistWords, st, s->sort_n, &tm, 3, 4));
    if (M >= (1ull << 32) - 65536 || s->Mb >= (1ull << 32) - 65536) return PVG_ERR_INSTANCE_OVERFLOW;
    s->M = M;
    if (block && M > 0) {   // the side stream is idle now: size and zero the block path's scratch beside the depth sort
      TRY(prep_block_bins(s, P, sd));
      CU(cudaEventRecord(s->ev_zero, sd));
    }
    // a2 scan: items per Gaussian = tiles (instances), or 8x8-tile blocks touched (block entries)
    TRY(run_scan(s, s->nv, block, block ? s->boffsets.as<uint32_t>() : s->offsets.as<uint32_t>(), visit, &tm, true));
    }
  } else {
    s->nv = n;
    TRY(run_scan(s, n, false, s->offsets.as<uint32_t>(), nullptr, &tm));
    CU(cudaMemcpyAsync(s->h_total, s->small.as<unsigned char>() + 8, 8, cudaMemcpyDeviceToHost, st));
    CU(cudaStreamSynchronize(st));   // index-order path: M is only known after the scan
    tm.cut();
    M = s->h_total[0];
  }
  if (M >= (1ull << 32) - 65536 || s->Mb >= (1ull << 32) - 65536) return PVG_ERR_INSTANCE_OVERFLOW;
  s->M = M;

  if (s->light && M == 0) {   // nothing survives: every record reads as zero
    CU(cudaMemsetAsync(s->record.p, 0, (size_t)n * 48, st));
    tm.cut();
    s->records_complete = true;
  }
  s->sorted_side = 0;
  const bool compact = !block && s->presort && s->compact && tile_bits <= 16;
  s->compact_used = compact;
  if (M > 0 && block) {
    CU(cudaStreamWaitEvent(st, s->ev_zero, 0));
    tm.cut();
    TRY(run_block_bins(s, P, visit, &tm));
  } else if (M > 0 && compact) {
    for (int k = 0; k < 2; ++k) {
      TRY(s->tiles16[k].reserve((size_t)M * 2, st, 1.125));
      TRY(s->vals[k].reserve((size_t)M * 4, st, 1.125));
    }
    TRY(tm.begin("duplicate", PVG_STAGE_DUPLICATE, st));
    expand_kernel<true><<<(unsigned)((M + EXP_CHUNK - 1) / EXP_CHUNK), EXP_THREADS, 0, st>>>(
        s->nv, (uint32_t)M, s->offsets.as<uint32_t>(), visit, s->tileinfo.as<uint4>(), (uint32_t)P.tiles_x, nullptr,
        s->tiles16[0].as<uint16_t>(), s->vals[0].as<uint32_t>());
    TRY(tm.end(st));
    if (s->keep_unsorted) {
      TRY(s->tiles16_unsorted.reserve((size_t)M * 2, st));
      TRY(s->vals_unsorted.reserve((size_t)M * 4, st));
      CU(cudaMemcpyAsync(s->tiles16_unsorted.p, s->tiles16[0].p, (size_t)M * 2, cudaMemcpyDeviceToDevice, st));
      CU(cudaMemcpyAsync(s->vals_unsorted.p, s->vals[0].p, (size_t)M * 4, cudaMemcpyDeviceToDevice, st));
      tm.cut();
    }
    int side = 0;
    TRY(run_compact_sort(s->dev, (uint32_t)M, s->tiles16[0].as<uint16_t>(), s->vals[0].as<uint32_t>(),
                         s->tiles16[1].as<uint16_t>(), s->vals[1].as<uint32_t>(), tile_bits, st, s->sort_m, &tm, &side));
    s->sorted_side = side;
  } else if (M > 0) {
    for (int k = 0; k < 2; ++k) {
      TRY(s->keys[k].reserve((size_t)M * 8, st, 1.125));
      TRY(s->vals[k].reserve((size_t)M * 4, st, 1.125));
    }
    // a2 emit
    TRY(tm.begin("duplicate", PVG_STAGE_DUPLICATE, st));
    expand_kernel<false><<<(unsigned)((M + EXP_CHUNK - 1) / EXP_CHUNK), EXP_THREADS, 0, st>>>(
        s->nv, (uint32_t)M, s->offsets.as<uint32_t>(), visit, s->tileinfo.as<uint4>(), (uint32_t)P.tiles_x,
        s->keys[0].as<uint64_t>(), nullptr, s->vals[0].as<uint32_t>());
    TRY(tm.end(st));
    if (s->keep_unsorted) {
      TRY(s->keys_unsorted.reserve((size_t)M * 8, st));
      TRY(s->vals_unsorted.reserve((size_t)M * 4, st));
      CU(cudaMemcpyAsync(s->keys_unsorted.p, s->keys[0].p, (size_t)M * 8, cudaMemcpyDeviceToDevice, st));
      CU(cudaMemcpyAsync(s->vals_unsorted.p, s->vals[0].p, (size_t)M * 4, cudaMemcpyDeviceToDevice, st));
      tm.cut();
    }
    // a3 (M-instance part)
    int side = 0;
    TRY(run_onesweep(s->dev, M, s->keys[0].as<uint64_t>(), s->vals[0].as<uint32_t>(), s->keys[1].as<uint64_t>(),
                     s->vals[1].as<uint32_t>(), s->sort_begin, s->sort_end, st, s->sort_m, &tm, PVG_STAGE_SORT, &side,
                     s->presort != 0));
    s->sorted_side = side;
    if (!s->presort) {
      // a4 ranges from the sorted keys
      TRY(tm.begin("tile_ranges", PVG_STAGE_RANGES, st));
      tile_ranges_kernel<<<(unsigned)((M + 255) / 256), 256, 0, st>>>(s->keys[side].as<uint64_t>(), M, tiles,
                                                                      s->ranges.as<uint2>());
      TRY(tm.end(st));
    }
  } else if (!s->presort) {
    CU(cudaMemsetAsync(s->ranges.p, 0, (size_t)tiles * 8, st));
    tm.cut();
  }

  // a5 blend
  TRY(tm.begin("blend", PVG_STAGE_BLEND, st));
  {
    unsigned long long* ctr = nullptr;
    if (s->count_pairs) {
      ctr = reinterpret_cast<unsigned long long*>(s->small.as<unsigned char>() + 64);
      CU(cudaMemsetAsync(ctr, 0, 16, st));
      tm.cut();
    }
    const uint2* rg = s->ranges.as<uint2>();
    const uint32_t* vl = s->vals[s->sorted_side].as<uint32_t>();
    const float4* rec = s->record.as<float4>();
    const int mode = P.target == 1 ? BLEND_FEATURE : (P.sky ? BLEND_SKY : BLEND_COLOR);
    const uint32_t band_tiles = (uint32_t)P.tiles_x * (uint32_t)(P.band_y1 - P.band_y0);
    const bool lazy = M > 0 && s->block_used && s->lazy_used;
    BlendLazy Z = {};
    if (lazy) {
      const size_t ntiles = (size_t)P.tiles_x * P.tiles_y;
      Z.state = s->lazy_state.as<float>();
      Z.unf_mask = s->unf.as<unsigned long long>();
      Z.unf_count = reinterpret_cast<uint32_t*>(s->unf.as<unsigned char>() + 2048);
      Z.lim = reinterpret_cast<const uint32_t*>(s->unf.as<unsigned char>() + kUnfHead);
      Z.unf_list = reinterpret_cast<uint32_t*>(s->unf.as<unsigned char>() + kUnfHead) + ntiles;
      Z.parked_host = s->d_total + 3;
      Z.blocks_x = bb_blocks(P.tiles_x);
    }
    R2Chain R2 = {};
    // Who launches the second round? The device, when the frame before parked nothing: then this one most likely parks
    // nothing either, and all the round costs is the one-thread gate. The host, when the frame before did park: grids
    // launched from the device ran far slower than the same kernels launched from the host (the second blend phase of
    // a frame whose 9600 tiles all park: 2.36 ms against 0.57 ms, the rest of the chain alike; a larger shared-memory
    // carve-out for the gate, whose configuration its children inherit, changed nothing), so a scene that does park
    // is better served by the host's launches, each of which looks at the parked count. Either way the frame is
    // complete and bit-identical; a wrong guess costs time only (4.3 ms instead of 2.2 ms for the all-parked frame,
    // 30 us of empty launches for a frame that parks nothing).
    if (lazy && PVG_R2_TAIL && PVG_BIN_FUSED && s->prev_parked == 0) TRY(fill_r2(s, P, band_tiles, &R2));
#define PVG_BLEND(C, M, PH) TRY(launch_chain(&tm, blend_kernel<C, M, PH>, dim3((PH) == 2 ? std::min(band_tiles, (uint32_t)s->dev.sms * 8u) : band_tiles), dim3(BLEND_THREADS), 0, st, P, rg, vl, rec, out_rgb, out_depth, out_alpha, ctr, (const float*)featw, Z))
#define PVG_BLEND_ALL(PH)                                        \
    if (s->count_pairs) {                                        \
      if (mode == BLEND_FEATURE) PVG_BLEND(true, BLEND_FEATURE, PH); \
      else if (mode == BLEND_SKY) PVG_BLEND(true, BLEND_SKY, PH);    \
      else PVG_BLEND(true, BLEND_COLOR, PH);                         \
    } else {                                                     \
      if (mode == BLEND_FEATURE) PVG_BLEND(false, BLEND_FEATURE, PH); \
      else if (mode == BLEND_SKY) PVG_BLEND(false, BLEND_SKY, PH);    \
      else PVG_BLEND(false, BLEND_COLOR, PH);                         \
    }
    if (!lazy) {
      PVG_BLEND_ALL(0)
    } else if (R2.enabled) {
      // the second round is launched from the device, by the gate, if a tile parked (round2.cu)
      PVG_BLEND_ALL(1)
      // with the timing hook on, an event record sits between the two kernels: a plain launch then
      const int pdl = (PVG_PDL && tm.pdl_open && tm.pdl_stream == st && !tm.frame_on) ? 1 : 0;
      TRY(tm.end(st));
      TRY(tm.begin("round2_gate", PVG_STAGE_BLEND, st));
      const int which = (s->count_pairs ? 3 : 0) + mode;
      const int e = pvg_r2_gate(s->dev.ordinal, (void*)st, &P, &R2, &Z, which, rg, vl, rec, out_rgb, out_depth, out_alpha, ctr,
                                (const float*)featw, pdl);
      if (e != 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "round2 gate: %s", cudaGetErrorString((cudaError_t)e));
        return PVG_ERR_CUDA;
      }
      tm.pdl_open = false;
      if (R2.back) s->nv = (uint32_t)s->survivors;
    } else {
      // phase 1 on the list prefixes; the tiles it could not finish get the rest of their lists, then phase 2
      PVG_BLEND_ALL(1)
      TRY(tm.end(st));
#if PVG_BIN_FUSED
      bool shading = false;
      if (s->emit_first < s->emit_tiles) {
        if (s->front_used && s->front < (uint32_t)s->survivors) {
          // front-first: the rest of the depth order and of the offsets, if a tile parked
          TRY(run_depth_back(s, Z.unf_count, &tm));
          s->nv = (uint32_t)s->survivors;
        }
        if (s->light) {
          // the rest of the scene's records, in index order (sequential model reads; the first slab's records are
          // rewritten with the same values), on the side stream: nothing before phase 2 of the blend needs them
          cudaStream_t sd = s->side;
          CU(cudaEventRecord(s->ev_fork, st));
          CU(cudaStreamWaitEvent(sd, s->ev_fork, 0));
          tm.cut();
          TRY(tm.begin("shade", PVG_STAGE_PREPROCESS, sd));
          TRY(run_shade_all(s, P, Z.unf_count, sd));
          TRY(tm.end(sd));
          CU(cudaEventRecord(s->ev_join, sd));
          shading = true;
        }
        TRY(tm.begin("bin_emit", PVG_STAGE_SORT, st));
        TRY(run_bin_emit(s, P, s->visit_last, s->emit_tiles - s->emit_first, Z.unf_count, true));
        TRY(tm.end(st));
      }
#endif
      TRY(tm.begin("bin_write", PVG_STAGE_SORT, st));
      TRY(launch_bin_write(s, P, (uint32_t)s->lazy_chunks, 0xFFFFFFFFu, true, 2));
      TRY(tm.end(st));
      if (shading) {
        CU(cudaStreamWaitEvent(st, s->ev_join, 0));
        tm.cut();
      }
      TRY(tm.begin("blend", PVG_STAGE_BLEND, st));
      PVG_BLEND_ALL(2)
    }
#undef PVG_BLEND_ALL
#undef PVG_BLEND
  }
  TRY(tm.end(st));
  CU(cudaGetLastError());
  s->rendered = true;
  return PVG_OK;
}

}  // namespace

extern "C" {

int pvg_version(void) { return 100; }

const char* pvg_strerror(int code) {
  switch (code) {
    case PVG_OK: return "ok";
    case PVG_ERR_NULL: return "null pointer argument";
    case PVG_ERR_BAD_DESC: return "bad scene descriptor";
    case PVG_ERR_BAD_CAMERA: return "bad camera";
    case PVG_ERR_OOM: return "device out of memory";
    case PVG_ERR_INSTANCE_OVERFLOW: return "tile instance count overflows 32 bits";
    case PVG_ERR_CUDA: return "CUDA error";
    case PVG_ERR_BAD_OPTION: return "bad option";
    case PVG_ERR_BAD_STATE: return "bad state (non-finite t or dt, negative rho_min, rho_max < rho_min)";
    case PVG_ERR_TOO_LARGE: return "too many pairs for the static scratch of pvg_sort_pairs_static";
    default: return "unknown error";
  }
}

const char* pvg_last_cuda_error(void) { return g_cuda_err; }

int pvg_set_allocator(pvg_alloc_fn alloc_fn, pvg_free_fn free_fn, void* user) {
  if ((alloc_fn == nullptr) != (free_fn == nullptr)) return PVG_ERR_NULL;
  g_alloc = alloc_fn;
  g_free = free_fn;
  g_alloc_user = user;
  return PVG_OK;
}

int pvg_set_stream(pvg_scene* scene, void* cuda_stream) {
  if (!scene) return PVG_ERR_NULL;
  cudaStream_t next = (cudaStream_t)cuda_stream;
  if (next == scene->stream) return PVG_OK;
  // The workspace (record, ranges, vals, histograms, ...) belongs to the frames already enqueued on the old
  // stream: the new stream -- and through ev_start / ev_rendered the side and copy streams -- must run behind them.
  DeviceGuard guard(scene->dev.ordinal);
  if (scene->ev_switch) {
    if (cudaEventRecord(scene->ev_switch, scene->stream) == cudaSuccess) {
      CU(cudaStreamWaitEvent(next, scene->ev_switch, 0));
    } else {   // the old stream is gone (destroyed by its owner): nothing finer to wait on
      cudaGetLastError();
      CU(cudaDeviceSynchronize());
    }
  }
  scene->stream = next;
  return PVG_OK;
}

int pvg_create_scene(const pvg_scene_desc* d, pvg_scene** out) {
  if (!d || !out) return PVG_ERR_NULL;
  *out = nullptr;
  if (!d->mu || !d->quat || !d->scale || !d->opacity || !d->sh || !d->tau || !d->beta || !d->vel) return PVG_ERR_NULL;
  if (d->n == 0 || d->n >= (1ull << 31)) return PVG_ERR_BAD_DESC;
  if (!(d->cycle > 0.f)) return PVG_ERR_BAD_DESC;  // also rejects NaN
  if (d->sh_degree < 0 || d->sh_degree > 3) return PVG_ERR_BAD_DESC;
  pvg_scene* s = new (std::nothrow) pvg_scene();
  if (!s) return PVG_ERR_OOM;
  const int rc = create_impl(d, s);
  if (rc != PVG_OK) {
    release_all(s);
    delete s;
    return rc;
  }
  *out = s;
  return PVG_OK;
}

int pvg_fork_scene(pvg_scene* scene, pvg_scene** out) {
  if (!scene || !out) return PVG_ERR_NULL;
  *out = nullptr;
  pvg_scene* s = new (std::nothrow) pvg_scene();
  if (!s) return PVG_ERR_OOM;
  DeviceGuard guard(scene->dev.ordinal);
  s->n = scene->n; s->cycle = scene->cycle; s->sh_degree = scene->sh_degree;
  s->stream = scene->stream;
  s->dev = scene->dev;
  s->presort = scene->presort; s->keep_unsorted = scene->keep_unsorted; s->count_pairs = scene->count_pairs;
  s->compact = scene->compact; s->block = scene->block; s->blend_cull = scene->blend_cull;
  s->lazy_chunks = scene->lazy_chunks; s->lazy_slab = scene->lazy_slab; s->exact_tiles = scene->exact_tiles; s->lazy_depth = scene->lazy_depth;
  s->band_begin = scene->band_begin; s->band_end = scene->band_end;
  s->timer.enabled = scene->timer.enabled; s->timer.accumulate = scene->timer.accumulate; s->timer.stride = scene->timer.stride;
  s->model = scene->model;
  s->model->refs.fetch_add(1);
  // the model was written on the parent's stream at creation, which synchronised: nothing to wait for
  const int rc = init_workspace(s);
  if (rc != PVG_OK) {
    release_all(s);
    delete s;
    return rc;
  }
  *out = s;
  return PVG_OK;
}

int pvg_destroy(pvg_scene* scene) {
  if (!scene) return PVG_ERR_NULL;
  DeviceGuard guard(scene->dev.ordinal);
  cudaStreamSynchronize(scene->stream);
  if (scene->side) cudaStreamSynchronize(scene->side);
  if (scene->copy_stream) cudaStreamSynchronize(scene->copy_stream);
  release_all(scene);
  delete scene;
  return PVG_OK;
}

int pvg_set_sky(pvg_scene* scene, const float* cube, int res, int on_device) {
  if (!scene) return PVG_ERR_NULL;
  DeviceGuard guard(scene->dev.ordinal);
  cudaStream_t st = scene->stream;
  CU(cudaStreamSynchronize(st));   // frames in flight may still read the old map
  if (scene->copy_stream) CU(cudaStreamSynchronize(scene->copy_stream));
  if (!cube) {
    scene->sky_res = 0;
    return PVG_OK;
  }
  if (res < 1 || res > 16384) return PVG_ERR_BAD_OPTION;
  const size_t bytes = (size_t)6 * res * res * 3 * sizeof(float);
  scene->sky_res = 0;
  TRY(scene->sky.reserve(bytes, st));
  CU(cudaMemcpyAsync(scene->sky.p, cube, bytes, on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, st));
  CU(cudaStreamSynchronize(st));
  scene->sky_res = res;
  return PVG_OK;
}

int pvg_set_option(pvg_scene* scene, int option, int64_t value) {
  if (!scene) return PVG_ERR_NULL;
  switch (option) {
    case PVG_OPT_PRESORT_DEPTH: scene->presort = value ? 1 : 0; return PVG_OK;
    case PVG_OPT_KEEP_UNSORTED: scene->keep_unsorted = value ? 1 : 0; return PVG_OK;
    case PVG_OPT_COMPACT_KEYS: scene->compact = value ? 1 : 0; return PVG_OK;
    case PVG_OPT_BLOCK_BINS: scene->block = value ? 1 : 0; return PVG_OK;
    case PVG_OPT_BLEND_CULL: scene->blend_cull = value ? 1 : 0; return PVG_OK;
    case PVG_OPT_COUNT_PAIRS: scene->count_pairs = value ? 1 : 0; return PVG_OK;
    case PVG_OPT_KERNEL_EVENTS:
      scene->timer.enabled = value != 0;
      scene->timer.accumulate = value == 2;
      scene->timer.renders = 0;
      scene->timer.reset();
      return PVG_OK;
    case PVG_OPT_LAZY_CHUNKS:
      if (value < 0 || value > (1 << 20)) return PVG_ERR_BAD_OPTION;
      scene->lazy_chunks = (int)value;
      return PVG_OK;
    case PVG_OPT_LAZY_SLAB:
      if (value < 1 || value > 4096) return PVG_ERR_BAD_OPTION;
      scene->lazy_slab = (int)value;
      return PVG_OK;
    case PVG_OPT_EXACT_TILES: scene->exact_tiles = value ? 1 : 0; return PVG_OK;
    case PVG_OPT_LAZY_DEPTH:
      if (value < 0 || value > 2) return PVG_ERR_BAD_OPTION;
      scene->lazy_depth = (int)value;
      return PVG_OK;
    case PVG_OPT_TILE_ROW_BEGIN:
      if (value < 0 || value > 2048) return PVG_ERR_BAD_OPTION;
      scene->band_begin = (int)value;
      return PVG_OK;
    case PVG_OPT_TILE_ROW_END:
      if (value < 0 || value > 2048) return PVG_ERR_BAD_OPTION;
      scene->band_end = (int)value;
      return PVG_OK;
    case PVG_OPT_EVENT_STRIDE:
      if (value < 1 || value > (1 << 20)) return PVG_ERR_BAD_OPTION;
      scene->timer.stride = (int)value;
      scene->timer.renders = 0;
      return PVG_OK;
    default: return PVG_ERR_BAD_OPTION;
  }
}

static bool state_ok(const pvg_state* st) {
  return std::isfinite(st->t) && std::isfinite(st->dt) && !(st->rho_min < 0.f) && !(st->rho_max < st->rho_min) &&
         (st->target == PVG_TARGET_COLOR || st->target == PVG_TARGET_DYNAMICS);
}

int pvg_render_state(pvg_scene* scene, const pvg_camera* cam, const pvg_state* state, float* out_rgb, float* out_depth,
                     float* out_alpha) {
  if (!scene || !cam || !state) return PVG_ERR_NULL;
  if (!state_ok(state)) return PVG_ERR_BAD_STATE;
  return render_impl(scene, cam, state, out_rgb, out_depth, out_alpha);
}

int pvg_render(pvg_scene* scene, const pvg_camera* cam, float t, float* out_rgb, float* out_depth, float* out_alpha) {
  const pvg_state st = {t, 0.f, 0.f, INFINITY, PVG_TARGET_COLOR};
  return pvg_render_state(scene, cam, &st, out_rgb, out_depth, out_alpha);
}

int pvg_wait_host(pvg_scene* scene) {
  if (!scene) return PVG_ERR_NULL;
  for (int k = 0; k < 2; ++k)
    if (scene->copy_pending[k]) {
      CU(cudaEventSynchronize(scene->ev_copied[k]));
      scene->copy_pending[k] = false;
    }
  return PVG_OK;
}

int pvg_render_host_async(pvg_scene* scene, const pvg_camera* cam, float t, float* host_rgb, float* host_depth,
                          float* host_alpha) {
  if (!scene || !cam) return PVG_ERR_NULL;
  const pvg_state state = {t, 0.f, 0.f, INFINITY, PVG_TARGET_COLOR};
  if (!state_ok(&state)) return PVG_ERR_BAD_STATE;
  if (cam->width <= 0 || cam->height <= 0 || cam->width > 32768 || cam->height > 32768) return PVG_ERR_BAD_CAMERA;
  const size_t HW = (size_t)cam->width * cam->height;
  DeviceGuard guard(scene->dev.ordinal);
  cudaStream_t st = scene->stream;
  const int slot = scene->img_next;
  scene->img_next ^= 1;
  // the frame rendered two calls ago used this device image: its copy must have left before the blend rewrites it
  if (scene->copy_pending[slot]) CU(cudaStreamWaitEvent(st, scene->ev_copied[slot], 0));
  if (HW * 5 * 4 > scene->img[slot].cap && scene->copy_pending[slot]) {   // growing frees the old buffer
    CU(cudaEventSynchronize(scene->ev_copied[slot]));
    scene->copy_pending[slot] = false;
  }
  TRY(scene->img[slot].reserve(HW * 5 * 4, st));
  float* d_rgb = scene->img[slot].as<float>();
  float* d_depth = d_rgb + 3 * HW;
  float* d_alpha = d_rgb + 4 * HW;
  TRY(render_impl(scene, cam, &state, host_rgb ? d_rgb : nullptr, host_depth ? d_depth : nullptr,
                  host_alpha ? d_alpha : nullptr));
  CU(cudaEventRecord(scene->ev_rendered, st));
  cudaStream_t cs = scene->copy_stream;
  CU(cudaStreamWaitEvent(cs, scene->ev_rendered, 0));
  if (host_rgb) CU(cudaMemcpyAsync(host_rgb, d_rgb, HW * 12, cudaMemcpyDeviceToHost, cs));
  if (host_depth) CU(cudaMemcpyAsync(host_depth, d_depth, HW * 4, cudaMemcpyDeviceToHost, cs));
  if (host_alpha) CU(cudaMemcpyAsync(host_alpha, d_alpha, HW * 4, cudaMemcpyDeviceToHost, cs));
  CU(cudaEventRecord(scene->ev_copied[slot], cs));
  scene->copy_pending[slot] = true;
  return PVG_OK;
}

int pvg_render_host(pvg_scene* scene, const pvg_camera* cam, float t, float* host_rgb, float* host_depth,
                    float* host_alpha) {
  TRY(pvg_render_host_async(scene, cam, t, host_rgb, host_depth, host_alpha));
  return pvg_wait_host(scene);
}

int pvg_debug_view(pvg_scene* s, pvg_debug* out) {
  if (!s || !out) return PVG_ERR_NULL;
  memset(out, 0, sizeof(*out));
  if (!s->rendered) return PVG_OK;
  DeviceGuard guard(s->dev.ordinal);
  s->timer.cut();
  out->n = s->n;
  out->num_instances = s->M;
  out->tiles_x = s->tiles_x;
  out->tiles_y = s->tiles_y;
  out->sort_begin_bit = (uint32_t)s->sort_begin;
  out->sort_end_bit = (uint32_t)s->sort_end;
  out->record = s->record.as<float>();
  out->counts = s->counts.as<uint32_t>();
  out->visit_order = s->presort_used ? s->dvals[s->visit_side].as<uint32_t>() : nullptr;
  out->offsets = s->offsets.as<uint32_t>();
  if (s->front_used && !s->depth_complete) {
    // front-first depth order: the frame ordered (and scanned) the back only if a tile parked -- the parked count of
    // the frame is in mapped host memory once the stream has drained
    CU(cudaStreamSynchronize(s->stream));
    if (s->M && s->front < (uint32_t)s->survivors && s->h_total[3] == 0) {
      TRY(run_depth_back(s, nullptr, nullptr));
      CU(cudaGetLastError());
    }
    s->nv = (uint32_t)s->survivors;
    s->depth_complete = true;
  }
  if (s->presort_used && s->nv < s->n && !s->visit_tail_done) {
    // The depth sort drops the culled Gaussians in its first pass: the frame's visiting order holds the S survivors.
    // The view documents all n positions (the culled ones follow, in index order): append them here, on the host --
    // a debugging call.
    std::vector<uint32_t> cnt(s->n), tail;
    CU(cudaStreamSynchronize(s->stream));
    CU(cudaMemcpy(cnt.data(), s->counts.p, (size_t)s->n * 4, cudaMemcpyDeviceToHost));
    tail.reserve(s->n - s->nv);
    for (uint32_t i = 0; i < s->n; ++i)
      if (cnt[i] == 0u) tail.push_back(i);
    if (tail.size() != (size_t)(s->n - s->nv)) {
      snprintf(g_cuda_err, sizeof(g_cuda_err), "debug view: %zu culled Gaussians, %u expected", tail.size(), s->n - s->nv);
      return PVG_ERR_CUDA;
    }
    CU(cudaMemcpy(s->dvals[s->visit_side].as<uint32_t>() + s->nv, tail.data(), tail.size() * 4, cudaMemcpyHostToDevice));
    s->visit_tail_done = true;
  }
  if (s->block_used && s->light && !s->records_complete && s->M) {
    // lazy lists: the records the frame never needed (and zeros for the culled Gaussians)
    TRY(run_shade_all(s, s->last_P, nullptr));
    CU(cudaGetLastError());
    s->records_complete = true;
  }
  if (s->block_used && s->lazy_used && !s->lists_complete && s->M) {
    // lazy lists: write what the frame never needed, so that vals_sorted is every tile's whole list
#if PVG_BIN_FUSED
    if (s->emit_first < s->emit_tiles) {
      // the entries behind the first slab, unless the frame's second round has formed them already (then the
      // ticket stands at emit_tiles; forming them twice would be harmless but the ticket must not run on)
      uint32_t tk = 0;
      CU(cudaMemcpyAsync(&tk, s->sort_m.tickets.as<uint32_t>(), 4, cudaMemcpyDeviceToHost, s->stream));
      CU(cudaStreamSynchronize(s->stream));
      if (tk < s->emit_tiles) TRY(run_bin_emit(s, s->last_P, s->visit_last, s->emit_tiles - tk, nullptr));
    }
#endif
    CU(cudaMemsetAsync(s->sort_m.tickets.as<uint32_t>() + 3, 0, 4, s->stream));
    TRY(launch_bin_write(s, s->last_P, (uint32_t)s->lazy_chunks_used, 0xFFFFFFFFu, false, 3));
    CU(cudaGetLastError());
    s->lists_complete = true;
  }
  if (s->block_used) {
    // the block path never forms per-instance offsets or the unsorted list: produce them here
    cudaStream_t st = s->stream;
    const uint32_t* visit = s->dvals[s->visit_side].as<uint32_t>();
    TRY(run_scan(s, s->n, false, s->offsets.as<uint32_t>(), visit, nullptr, false,
                 s->exact_used ? s->counts_exact.as<uint32_t>() : nullptr));
    if (s->M) {
      TRY(s->keys[0].reserve((size_t)s->M * 8, st));
      keys_from_ranges_kernel<<<s->tiles_x * s->tiles_y, 256, 0, st>>>(s->ranges.as<uint2>(), s->vals[0].as<uint32_t>(),
                                                                        s->tileinfo.as<uint4>(), s->keys[0].as<uint64_t>());
      if (s->keep_unsorted_used && !s->exact_used) {   // (the exact lists have no unsorted form: their masks are refined after the split)
        TRY(s->keys_unsorted.reserve((size_t)s->M * 8, st));
        TRY(s->vals_unsorted.reserve((size_t)s->M * 4, st));
        expand_kernel<false><<<(unsigned)((s->M + EXP_CHUNK - 1) / EXP_CHUNK), EXP_THREADS, 0, st>>>(
            s->n, (uint32_t)s->M, s->offsets.as<uint32_t>(), visit, s->tileinfo.as<uint4>(), s->tiles_x,
            s->keys_unsorted.as<uint64_t>(), nullptr, s->vals_unsorted.as<uint32_t>());
      }
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
  }
  if (s->compact_used && s->M) {
    // rebuild (tile << 32 | depth bits) from the compact payload: debug only
    cudaStream_t st = s->stream;
    const uint32_t M32 = (uint32_t)s->M;
    TRY(s->keys[0].reserve((size_t)s->M * 8, st));
    keys_from_ranges_kernel<<<s->tiles_x * s->tiles_y, 256, 0, st>>>(s->ranges.as<uint2>(),
                                                                      s->vals[s->sorted_side].as<uint32_t>(),
                                                                      s->tileinfo.as<uint4>(), s->keys[0].as<uint64_t>());
    if (s->keep_unsorted_used) {
      TRY(s->keys_unsorted.reserve((size_t)s->M * 8, st));
      keys_from_tiles16_kernel<<<(M32 + 255) / 256, 256, 0, st>>>(s->tiles16_unsorted.as<uint16_t>(),
                                                                 s->vals_unsorted.as<uint32_t>(), s->tileinfo.as<uint4>(),
                                                                 M32, s->keys_unsorted.as<uint64_t>());
    }
    CU(cudaGetLastError());
    CU(cudaStreamSynchronize(st));
  }
  if (s->keep_unsorted_used && s->M && !s->exact_used) {
    out->keys_unsorted = s->keys_unsorted.as<uint64_t>();
    out->vals_unsorted = s->vals_unsorted.as<uint32_t>();
  }
  if (s->M) {
    out->keys_sorted = s->keys[(s->compact_used || s->block_used) ? 0 : s->sorted_side].as<uint64_t>();
    out->vals_sorted = s->vals[s->sorted_side].as<uint32_t>();
  }
  out->ranges = s->ranges.as<uint32_t>();
  if (s->exact_used) {   // the exact lists: their own counts and total (the stream was synchronised above)
    out->counts = s->counts_exact.as<uint32_t>();
    out->num_instances = s->M ? s->h_total[7] : 0;
  }
  return PVG_OK;
}

int pvg_kernel_times_ms(pvg_scene* s, int cap, const char** names, int* stages, float* ms) {
  if (!s) return PVG_ERR_NULL;
  if (!s->rendered || !s->timer.enabled) return 0;
  CU(cudaStreamSynchronize(s->stream));
  const int cnt = (int)s->timer.recs.size();
  for (int i = 0; i < cnt && i < cap; ++i) {
    const KernelRec& r = s->timer.recs[i];
    float v = 0.f;
    CU(cudaEventElapsedTime(&v, r.e0, r.e1));
    if (names) names[i] = r.name;
    if (stages) stages[i] = r.stage;
    if (ms) ms[i] = v;
  }
  if (s->timer.accumulate) s->timer.reset();
  return cnt;
}

int pvg_kernel_timeline_ms(pvg_scene* s, int cap, const char** names, float* start_ms, float* dur_ms) {
  if (!s) return PVG_ERR_NULL;
  if (!s->rendered || !s->timer.enabled || s->timer.recs.empty()) return 0;
  CU(cudaStreamSynchronize(s->stream));
  if (s->side) CU(cudaStreamSynchronize(s->side));
  const int cnt = (int)s->timer.recs.size();
  const cudaEvent_t origin = s->timer.recs[0].e0;
  for (int i = 0; i < cnt && i < cap; ++i) {
    const KernelRec& r = s->timer.recs[i];
    float a = 0.f, d = 0.f;
    CU(cudaEventElapsedTime(&a, origin, r.e0));
    CU(cudaEventElapsedTime(&d, r.e0, r.e1));
    if (names) names[i] = r.name;
    if (start_ms) start_ms[i] = a;
    if (dur_ms) dur_ms[i] = d;
  }
  return cnt;
}

int pvg_stage_times_ms(pvg_scene* s, float ms[PVG_NUM_STAGES]) {
  if (!s || !ms) return PVG_ERR_NULL;
  for (int k = 0; k < PVG_NUM_STAGES; ++k) ms[k] = 0.f;
  if (!s->rendered || !s->timer.enabled) return PVG_OK;
  CU(cudaStreamSynchronize(s->stream));
  // a stage runs from its first launch to its last one's end (includes memsets and the M read-back)
  for (int k = 0; k < PVG_NUM_STAGES; ++k) {
    const KernelRec *first = nullptr, *last = nullptr;
    for (const KernelRec& r : s->timer.recs)
      if (r.stage == k) { if (!first) first = &r; last = &r; }
    if (first) CU(cudaEventElapsedTime(&ms[k], first->e0, last->e1));
  }
  return PVG_OK;
}

int pvg_frame_stats(pvg_scene* s, uint64_t out[10]) {
  if (!s || !out) return PVG_ERR_NULL;
  out[0] = s->n;
  out[1] = s->rendered ? s->M : 0;
  out[2] = s->tiles_x;
  out[3] = s->tiles_y;
  out[4] = s->rendered ? s->Mb : 0;
  out[5] = s->block_used ? (s->exact_used ? 3 : 2) : (s->compact_used ? 1 : 0);
  out[6] = (s->rendered && s->presort_used) ? s->survivors : 0;
  // tiles the lazy lists' first blend phase parked (stored by the second phase through mapped host memory: it is
  // the last frame's figure once that frame has completed on the stream; the word is only read here)
  out[7] = (s->rendered && s->block_used && s->lazy_used && s->M) ? s->h_total[3] : 0;
  // exact lists: the instances actually listed (stored by exact_ranges_kernel through mapped host memory: the last
  // frame's figure once that frame has completed on the stream)
  out[8] = (s->rendered && s->exact_used && s->M) ? s->h_total[7] : 0;
  out[9] = (s->rendered && s->front_used) ? s->front : 0;   // front-first depth order: the pairs ordered up front
  return PVG_OK;
}

int pvg_blend_counters(pvg_scene* s, uint64_t out[2]) {
  if (!s || !out) return PVG_ERR_NULL;
  out[0] = out[1] = 0;
  if (!s->rendered || !s->count_pairs) return PVG_OK;
  CU(cudaStreamSynchronize(s->stream));
  CU(cudaMemcpy(out, s->small.as<unsigned char>() + 64, 16, cudaMemcpyDeviceToHost));
  return PVG_OK;
}

int pvg_calibrate_fp32(int mode, void* cuda_stream, double* thread_instr_per_s, int* sm_count) {
  if (!thread_instr_per_s) return PVG_ERR_NULL;
  if (mode < 0 || mode > 2) return PVG_ERR_BAD_OPTION;
  Dev dv;
  TRY(dv.query());
  if (sm_count) *sm_count = dv.sms;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const unsigned grid = (unsigned)dv.sms * 8u;   // 8 CTAs of 256 threads per SM: 16 warps per scheduler
  const int trips = 4096;
  float* sink = nullptr;
  CU(cudaMalloc(&sink, (size_t)grid * CALIB_THREADS * sizeof(float)));
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int rc = PVG_OK;
  float best = 0.f;
  do {
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) { rc = PVG_ERR_CUDA; break; }
    for (int rep = 0; rep < 6 && rc == PVG_OK; ++rep) {   // first launches warm up; the best of the rest counts
      cudaEventRecord(e0, st);
      if (mode == 0) calib_kernel<0><<<grid, CALIB_THREADS, 0, st>>>(sink, trips, 0.999f, 1e-3f, 0x5bd1e995u, 0x1b873593u);
      else if (mode == 1) calib_kernel<1><<<grid, CALIB_THREADS, 0, st>>>(sink, trips, 0.999f, 1e-3f, 0x5bd1e995u, 0x1b873593u);
      else calib_kernel<2><<<grid, CALIB_THREADS, 0, st>>>(sink, trips, 0.999f, 1e-3f, 0x5bd1e995u, 0x1b873593u);
      cudaEventRecord(e1, st);
      float ms = 0.f;
      if (cudaEventSynchronize(e1) != cudaSuccess || cudaEventElapsedTime(&ms, e0, e1) != cudaSuccess) { rc = PVG_ERR_CUDA; break; }
      if (rep >= 2 && ms > 0.f && (best == 0.f || ms < best)) best = ms;
    }
  } while (false);
  if (rc != PVG_OK) snprintf(g_cuda_err, sizeof(g_cuda_err), "calibrate: %s", cudaGetErrorString(cudaGetLastError()));
  if (e0) cudaEventDestroy(e0);
  if (e1) cudaEventDestroy(e1);
  cudaFree(sink);
  if (rc == PVG_OK) *thread_instr_per_s = best > 0.f ? calib_instructions(mode, grid, trips) / ((double)best * 1e-3) : 0.0;
  return rc;
}

int pvg_guard_bands(int enable) {
  g_guards.store(enable != 0);
  return PVG_OK;
}

int pvg_check_guards(uint64_t* damaged_allocations, uint64_t* checked_allocations) {
  CU(cudaDeviceSynchronize());
  std::lock_guard<std::mutex> lk(g_guard_mu);
  std::vector<unsigned char> h(kGuard);
  uint64_t bad = 0;
  for (const auto& kv : g_guarded) {
    const unsigned char* user = static_cast<const unsigned char*>(kv.first);
    bool ok = true;
    for (int side = 0; side < 2 && ok; ++side) {
      CU(cudaMemcpy(h.data(), side ? user + kv.second : user - kGuard, kGuard, cudaMemcpyDeviceToHost));
      for (size_t i = 0; i < kGuard; ++i)
        if (h[i] != (unsigned char)kGuardByte) { ok = false; break; }
    }
    if (!ok) ++bad;
  }
  if (damaged_allocations) *damaged_allocations = bad;
  if (checked_allocations) *checked_allocations = g_guarded.size();
  return PVG_OK;
}

int pvg_memcpy_d2h(void* host_dst, const void* device_src, size_t bytes) {
  if (bytes && (!host_dst || !device_src)) return PVG_ERR_NULL;
  if (bytes) CU(cudaMemcpy(host_dst, device_src, bytes, cudaMemcpyDeviceToHost));
  return PVG_OK;
}

int pvg_sort_pairs(uint64_t n, uint64_t* keys_in, uint32_t* vals_in, uint64_t* keys_out, uint32_t* vals_out,
                   int begin_bit, int end_bit, void* cuda_stream) {
  if (n && (!keys_in || !vals_in || !keys_out || !vals_out)) return PVG_ERR_NULL;
  if (begin_bit < 0 || end_bit > 64 || begin_bit > end_bit) return PVG_ERR_BAD_OPTION;
  if (n >= (1ull << 32)) return PVG_ERR_INSTANCE_OVERFLOW;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  SortScratch sc;
  int side = 0;
  Dev dv;
  TRY(dv.query());
  int rc = run_onesweep(dv, n, keys_in, vals_in, keys_out, vals_out, begin_bit, end_bit, st, sc, nullptr, 0, &side);
  if (rc == PVG_OK && n && side == 0) {  // result landed in the input buffers
    cudaError_t e = cudaMemcpyAsync(keys_out, keys_in, n * 8, cudaMemcpyDeviceToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(vals_out, vals_in, n * 4, cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) { snprintf(g_cuda_err, sizeof(g_cuda_err), "sort copy: %s", cudaGetErrorString(e)); rc = PVG_ERR_CUDA; }
  }
  cudaError_t e = cudaStreamSynchronize(st);
  if (rc == PVG_OK && e != cudaSuccess) { snprintf(g_cuda_err, sizeof(g_cuda_err), "sort: %s", cudaGetErrorString(e)); rc = PVG_ERR_CUDA; }
  sc.hist.release(); sc.lookback.release(); sc.tickets.release();
  return rc;
}

}  // extern "C"

// ---- the sort primitive without any allocation ---------------------------------------------------------------------
// pvg_sort_pairs sizes its scratch (digit histograms, tickets, look-back words) with the device allocator on every
// call. Callers that may not allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc -- get the same sort with that scratch in a file-scope device array of a fixed, modest size: every GPU that
// loads the library holds these 4.01 MB until the process exits. The array's name is a host-side stand-in in host
// code, not a device address: the address is looked up once per device (cudaGetSymbolAddress, with that device current).
constexpr uint64_t kSortStaticMaxN = PVG_SORT_STATIC_MAX_N;
constexpr size_t kSsTile = (size_t)OsSmall::THREADS * OsSmall::ITEMS;
constexpr size_t kSsTiles = (kSortStaticMaxN + kSsTile - 1) / kSsTile;
constexpr size_t kSsHistBytes = (size_t)OS_MAX_PASSES * OS_RADIX * 4;                  // 10 KB
constexpr size_t kSsTicketBytes = 256;                                                  // OS_MAX_PASSES u32, padded
constexpr size_t kSsLookbackBytes = (size_t)8 * kSsTiles * OS_RADIX * 8;                // at most 8 passes of 8 bits for 64 key bits
constexpr size_t kSsBytes = kSsHistBytes + kSsTicketBytes + kSsLookbackBytes;
static_assert(kSortStaticMaxN < OS_SMALL_BELOW, "the static scratch is laid out for the small tile shape");
static_assert(kSsHistBytes % 256 == 0 && OS_MAX_PASSES * 4 <= kSsTicketBytes, "aligned sections");
static __device__ __align__(256) unsigned char g_sort_static_scratch[kSsBytes];

namespace {
std::mutex g_ss_mu;
void* g_ss_ptr[64] = {};   // device address of g_sort_static_scratch, per device ordinal

int sort_static_scratch(int device, unsigned char** out) {
  if (device < 0 || device >= 64) return PVG_ERR_BAD_OPTION;
  std::lock_guard<std::mutex> lk(g_ss_mu);
  if (!g_ss_ptr[device]) {
    void* ptr = nullptr;
    CU(cudaGetSymbolAddress(&ptr, g_sort_static_scratch));   // the current device's copy (Dev::query read the ordinal just now)
    if (!ptr) {
      snprintf(g_cuda_err, sizeof(g_cuda_err), "sort scratch: cudaGetSymbolAddress returned a null address");
      return PVG_ERR_CUDA;
    }
    g_ss_ptr[device] = ptr;
  }
  *out = static_cast<unsigned char*>(g_ss_ptr[device]);
  return PVG_OK;
}
}  // namespace

extern "C" {

uint64_t pvg_sort_pairs_static_max_n(void) { return kSortStaticMaxN; }

int pvg_sort_pairs_static(uint64_t n, uint64_t* keys_in, uint32_t* vals_in, uint64_t* keys_out, uint32_t* vals_out,
                          int begin_bit, int end_bit, void* cuda_stream) {
  if (n && (!keys_in || !vals_in || !keys_out || !vals_out)) return PVG_ERR_NULL;
  if (begin_bit < 0 || end_bit > 64 || begin_bit > end_bit) return PVG_ERR_BAD_OPTION;
  if (n > kSortStaticMaxN) {
    snprintf(g_cuda_err, sizeof(g_cuda_err), "pvg_sort_pairs_static: n = %llu exceeds the static scratch (at most %llu pairs)",
             (unsigned long long)n, (unsigned long long)kSortStaticMaxN);
    return PVG_ERR_TOO_LARGE;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  Dev dv;
  TRY(dv.query());
  unsigned char* base = nullptr;
  TRY(sort_static_scratch(dv.ordinal, &base));
  // views of the static array: never reserved, grown or released (cap is what the array holds)
  SortScratch sc;
  sc.hist.p = base;                                   sc.hist.cap = kSsHistBytes;
  sc.tickets.p = base + kSsHistBytes;                 sc.tickets.cap = kSsTicketBytes;
  sc.lookback.p = base + kSsHistBytes + kSsTicketBytes; sc.lookback.cap = kSsLookbackBytes;
  int side = 0;
  if (n && end_bit > begin_bit) {
    // the array keeps the last call's contents: what must start at zero is cleared here, on the caller's stream
    const SortPlan plan = make_sort_plan(begin_bit, end_bit);
    const size_t tiles = ((size_t)n + kSsTile - 1) / kSsTile;
    const size_t lb_bytes = (size_t)plan.num_passes * tiles * OS_RADIX * 8;
    if (plan.num_passes > 8 || lb_bytes > kSsLookbackBytes) return PVG_ERR_TOO_LARGE;
    CU(cudaMemsetAsync(sc.hist.p, 0, kSsHistBytes + kSsTicketBytes, st));
    CU(cudaMemsetAsync(sc.lookback.p, 0, lb_bytes, st));
    TRY(run_onesweep(dv, n, keys_in, vals_in, keys_out, vals_out, begin_bit, end_bit, st, sc, nullptr, 0, &side, false, true));
  }
  if (n && side == 0) {   // result landed in the input buffers (an even number of passes, or none)
    CU(cudaMemcpyAsync(keys_out, keys_in, n * 8, cudaMemcpyDeviceToDevice, st));
    CU(cudaMemcpyAsync(vals_out, vals_in, n * 4, cudaMemcpyDeviceToDevice, st));
  }
  return PVG_OK;
}

}  // extern "C"
