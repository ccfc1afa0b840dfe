// mcrt.cu -- C-ABI boundary (include/mcrt.h) of the sm_100a Monte Carlo radiative-transfer path.
// Host code here only validates arguments, owns device memory and launches kernels; every step
// of the method (table build, emission, walk, interactions, tallies, temperature update) runs in
// the kernels of transport.cuh / tables.cuh.  There is no CPU fallback.
#include "mcrt.h"
#include "mcrt_dev.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "calibrate.cuh"
#include "tables.cuh"
#include "transport.cuh"
#include "transport_u.cuh"
#include "pah.cuh"

using namespace mcrt;

// ---- device memory of the library: a small caching allocator ---------------------------------------------------
// A job allocates ~25 device arrays in its set-up calls; cudaMalloc / cudaFree cost 40 us apiece on one box and
// 250 us on another (setup_ms 1.0 ... 6.3 in bench.py's e2e).  Blocks of up to 256 MB that a context gives back are
// kept (at most 1 GB in all) and handed out again to the next request of exactly the same size -- a second job
// of the same shape allocates nothing.  mc_free synchronises the device like cudaFree does, so a block is never
// handed on while a kernel may still use it.
#include <map>
#include <mutex>
namespace {
// Process-lifetime singletons, never destroyed: a context may be destroyed (Python's Context.__del__) after the
// static destructors of this library have run.
struct McBlock { int device; size_t bytes; };
struct McState {
  std::mutex mutex;
  std::multimap<std::pair<int, size_t>, void*> cache;         // (owning device, bytes) -> block
  size_t cached = 0;
  std::map<void*, McBlock> live;                              // every block of the library: the device it was allocated on
};
McState& mc_state() { static McState* s = new McState; return *s; }
constexpr size_t kMcBlockMax = (size_t)256 << 20, kMcTotalMax = (size_t)1 << 30;

// Makes `dev` the current device for its lifetime (blocks are synchronised and freed on the device that owns them).
struct DeviceScope {
  int prev = -1; bool switched = false;
  explicit DeviceScope(int dev) {
    if (cudaGetDevice(&prev) == cudaSuccess && prev != dev && dev >= 0) switched = cudaSetDevice(dev) == cudaSuccess;
  }
  ~DeviceScope() { if (switched) cudaSetDevice(prev); }
};

// While one of these is alive on a thread, mc_free on that thread skips its device synchronisation: the caller has
// synchronised the device itself and launches nothing until the scope ends (mcrt_destroy: one wait, not one per block).
thread_local int tl_mc_device_idle = 0;
struct DeviceIdleScope {
  DeviceIdleScope() { ++tl_mc_device_idle; }
  ~DeviceIdleScope() { --tl_mc_device_idle; }
};

// Frees every cached block (the caller holds the lock).
size_t mc_release_cache_locked(McState& S) {
  const size_t bytes = S.cached;
  for (auto& kv : S.cache) {
    DeviceScope scope(kv.first.first);
    S.live.erase(kv.second);
    cudaFree(kv.second);
  }
  S.cache.clear();
  S.cached = 0;
  return bytes;
}
}  // namespace
template <typename T>
static cudaError_t mc_malloc(T** p, size_t bytes) {
  McState& S = mc_state();
  int dev = 0;
  const bool have_dev = cudaGetDevice(&dev) == cudaSuccess;
  if (bytes && bytes <= kMcBlockMax && have_dev) {
    std::lock_guard<std::mutex> lock(S.mutex);
    auto it = S.cache.find({dev, bytes});
    if (it != S.cache.end()) {
      *p = static_cast<T*>(it->second);
      S.cache.erase(it);
      S.cached -= bytes;
      return cudaSuccess;
    }
  }
  void* q = nullptr;
  cudaError_t e = cudaMalloc(&q, bytes);
  if (e == cudaErrorMemoryAllocation) {                      // give the cache back and try once more
    (void)cudaGetLastError();
    {
      std::lock_guard<std::mutex> lock(S.mutex);
      mc_release_cache_locked(S);
    }
    e = cudaMalloc(&q, bytes);
  }
  if (e == cudaSuccess) {
    *p = static_cast<T*>(q);
    std::lock_guard<std::mutex> lock(S.mutex);
    S.live[q] = McBlock{have_dev ? dev : -1, bytes};
  }
  return e;
}
static cudaError_t mc_free(void* q) {
  if (!q) return cudaSuccess;
  McState& S = mc_state();
  McBlock blk{-1, 0};
  {
    std::lock_guard<std::mutex> lock(S.mutex);
    auto it = S.live.find(q);
    if (it != S.live.end()) blk = it->second;
  }
  DeviceScope scope(blk.device);                             // the device the block lives on, whichever is current
  if (blk.bytes && blk.bytes <= kMcBlockMax && blk.device >= 0) {
    if (!tl_mc_device_idle) cudaDeviceSynchronize();
    std::lock_guard<std::mutex> lock(S.mutex);
    if (S.cached + blk.bytes <= kMcTotalMax) {
      S.cache.insert({{blk.device, blk.bytes}, q});
      S.cached += blk.bytes;
      return cudaSuccess;
    }
  }
  {
    std::lock_guard<std::mutex> lock(S.mutex);
    S.live.erase(q);
  }
  return cudaFree(q);
}

// ---- device array of mcrt_get_cell_temperature_noalloc (include/mcrt.h) -------------------------------------------
// Part of the library image: every GPU that loads the library holds these 4 MiB until the process exits.  The
// name below is only a handle in host code -- it is NOT a device address there; the address of a GPU's copy comes
// from cudaGetSymbolAddress with that GPU current (noalloc_T_array, once per GPU).
constexpr long long kNoallocMaxSlots = MCRT_NOALLOC_MAX_SLOTS;
static __device__ __align__(256) float g_noalloc_T[kNoallocMaxSlots];
constexpr int kNoallocMaxDevices = 64;
static float* g_noalloc_T_ptr[kNoallocMaxDevices] = {};      // [device] address of that GPU's copy; nullptr: not asked yet
static std::mutex g_noalloc_mutex;                           // one call at a time: the array is shared

struct BatchEvents { cudaEvent_t e0, e1, e2; };

struct mcrt_ctx {
  int device = 0, sm_count = 0;
  int N = 0, S = 1;
  long long n3 = 0, n_ref = 0, slots = 0;
  long long store_n3 = 0;                 // storage slots of the root grid (sub-cells follow it)
  double origin[3] = {0, 0, 0}, root_size = 1;
  float* d_rho = nullptr;
  float* d_lnrho = nullptr;               // ln of d_rho (-inf: empty leaf / refined-cube marker), for the temperature update
  unsigned long long* d_tally = nullptr;
  float* d_trow = nullptr;
  // opacity
  int nb = 0, nT = 0;
  double Tmin = 1, Tmax = 1e4, dlnT = 0;
  double *d_nu = nullptr, *d_dnu = nullptr, *d_kabs = nullptr;
  float4* d_opac = nullptr;
  float *d_lnQ = nullptr, *d_cdf = nullptr;
  int* d_guide = nullptr;                 // [kGuide] bracket guide of the ln Q table (tables.cuh)
  uint32_t* d_cdf_guide = nullptr;        // [nT][kCdfGuide] bracket guide of the emission rows (tables.cuh)
  int cdf_guide_off = 0;                  // mcrt_set_cdf_guide(0): plain bisection (for the bit-identity test)
  // sources
  int nsrc = 0;
  SrcDev* d_src = nullptr;
  double* d_csrc = nullptr;               // [nsrc][nb] fp64 source CDFs (emission decisions are exact)
  float* d_csrc32 = nullptr;              // ... and their fp32 copy
  double Ltot = 0;
  // tallies: [0] work-queue head, [1..CNT_N] counters, then sed[3*nb], emit_bin[nb]
  unsigned long long* d_small = nullptr;
  unsigned long long* d_heads = nullptr;  // two work-queue heads used in turn: a launch zeroes the one its successor takes
  int head = 0;
  const void* occ_kern = nullptr;         // launch set-up of the transport kernel done for this (kernel, threads, bytes)
  int occ_threads = 0, occ_resident = 0;
  size_t occ_smem = 0;
  unsigned long long Ncum = 0;            // packages this context has transported since the last reset
  unsigned long long Nglobal = 0;         // packages of ALL ranks behind the temperatures (= Ncum on one GPU)
  cudaStream_t last_stream = nullptr;
  std::vector<BatchEvents> pending, spare;
  // single-level grids: storage layout (transport_u.cuh); `slots` stays the caller-visible count
  bool uni = false;
  LayoutU lay = {0, 0, 0, 0};
  // Macro cubes (single-level grids whose density is piecewise uniform): internally the grid is run as a
  // two-level one -- N/M macro cubes per axis, each with its M^3 cells behind the macro array; a macro cube
  // whose cells all hold the same density is walked in ONE step (transport_u.cuh, MACRO).  N, S, root_size
  // then describe the macro grid; n_fine / lay_fine the caller's grid (the getters' slot order, R22).
  int macro = 0, n_fine = 0;
  LayoutU lay_fine = {0, 0, 0, 0};
  long long store_slots = 0;
  int* d_lut = nullptr;
  unsigned long long* d_tally_scratch = nullptr;
  uint32_t* d_perm = nullptr;             // package numbers of a batch grouped by source
  unsigned long long perm_cap = 0;
  bool group_smem_set = false;            // k_group_by_source may use more than 48 KB of shared memory
  uint16_t* d_keys = nullptr;             // group of every package of the batch (kept between the two grouping passes)
  unsigned long long keys_cap = 0;
  unsigned int* d_srccnt = nullptr;       // [2][nsrc] counts, cursors
  int order_by_source = -1;               // -1 automatic, 0 off, 1 by source, 2 by source and start direction
  void* d_out_scratch = nullptr;          // staging for host read-outs that need a conversion kernel (8 B x slots)
  int quorum = 0;                         // 0 = automatic (from the job's crossings per flight so far)
  int tail_mode = -1;                     // end of a batch: -1 automatic (= 3); bit 0: the quorum follows the live lanes;
                                          // bit 1: the temperature update runs at the end of the transport launch
  int coop_launch = 0;                    // the device launches kernels cooperatively (grid-wide barrier)
  // region sweeps (transport_u.cuh, REGION): single-level bricked grids far larger than the L2
  int region_cells[3] = {0, 0, 0};        // cells per region along x, y, z (0: the grid does not qualify)
  int region_sweeps = -1;                 // -1 automatic, 0 off
  int *d_lut_marked = nullptr, *d_lut_plain2 = nullptr;     // [12 N]: marked | plain root tables; plain | plain
  float4* d_rec = nullptr;                // [perm_cap][3] suspended packages
  unsigned long long* d_list[2] = {nullptr, nullptr};       // suspended packages of a sweep: region << 32 | number
  unsigned int* d_swcnt = nullptr;        // [kMaxSweeps + 2] packages suspended in each sweep
  unsigned int* d_regcnt = nullptr;       // [2][regions] histogram, cursors
  unsigned long long rec_cap = 0;
  // density staged in shared memory (single-level grids): 0 none, 1 the fp32 array itself, 2 one bit per slot
  int dens_mode = 0, dens_off = 0;        // dens_off: the caller switched staging off (mcrt_set_density_staging)
  uint32_t* d_bits = nullptr;
  unsigned stage_bytes = 0;
  float pal0 = 0.f, pal1 = 0.f;
  int threads = 256, blocks_per_sm = 0;   // 0 = automatic (5; 4 on HBM-resident single-level grids)
  long long launches = 0;
  // observer (O9 / R34): escape-direction tallies, off by default
  ObserverDev obs = {0, 0, 0, -1, {0, 0, 1}, {1, 0, 0}, {0, 1, 0}, 1.f, 1.f, nullptr, nullptr};
  // asynchronous read-out (mcrt_results_begin / _wait): two tickets, each with its own device snapshot,
  // pinned staging of the small tallies and events; copies run on the context's own stream
  struct Ticket {
    bool busy = false;
    unsigned long long* snap_abs = nullptr; float* snap_T = nullptr; unsigned long long* snap_small = nullptr;
    unsigned long long* h_small = nullptr;                  // pinned
    cudaEvent_t ev_snap = nullptr, ev_done = nullptr;
    mcrt_counters* counters = nullptr; uint64_t* emitted = nullptr; uint64_t* sed = nullptr; mcrt_mem mem = MCRT_HOST;
  } tickets[2];
  int next_ticket = 0;
  cudaStream_t copy_stream = nullptr;
  // transiently heated PAH (row f2, pah.cuh): tables and the per-leaf, per-bin tallies / emission CDFs
  bool pah = false;
  PahDev pahd = {};
  double *d_kabs_eq = nullptr, *d_pah_C = nullptr, *d_pah_E = nullptr, *d_pah_T = nullptr, *d_pah_U = nullptr,
         *d_pah_Lam = nullptr, *d_pah_W = nullptr, *d_pah_P = nullptr;
  int* d_pah_J = nullptr;
  unsigned long long* d_pah_next = nullptr;   // work-queue head of k_pah_update
  float *d_pah_q = nullptr, *d_pah_cdf = nullptr, *d_pah_cold = nullptr, *d_pah_W32 = nullptr;
  uint32_t* d_pah_cnt = nullptr;
  bool have_opacity = false, have_source = false;
  std::string err;
};

static thread_local std::string g_err;   // errors raised without a context (per calling thread)

static mcrt_status fail(mcrt_ctx* c, mcrt_status st, const std::string& msg) {
  if (c) c->err = msg; else g_err = msg;
  return st;
}
#define CU(call)                                                                          \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess)                                                                \
      return fail(ctx, e_ == cudaErrorMemoryAllocation ? MCRT_ENOMEM : MCRT_ECUDA,        \
                  std::string(#call) + ": " + cudaGetErrorString(e_));                    \
  } while (0)

static void free_opacity(mcrt_ctx* c) {
  mc_free(c->d_nu); mc_free(c->d_dnu); mc_free(c->d_kabs); mc_free(c->d_opac);
  mc_free(c->d_lnQ); mc_free(c->d_cdf); mc_free(c->d_small); mc_free(c->d_guide); mc_free(c->d_cdf_guide);
  c->d_cdf_guide = nullptr;
  c->d_nu = c->d_dnu = c->d_kabs = nullptr; c->d_opac = nullptr; c->d_lnQ = c->d_cdf = nullptr; c->d_guide = nullptr;
  c->d_small = nullptr;
}
static void free_pah(mcrt_ctx* c) {
  mc_free(c->d_kabs_eq); mc_free(c->d_pah_C); mc_free(c->d_pah_E); mc_free(c->d_pah_T); mc_free(c->d_pah_U);
  mc_free(c->d_pah_Lam); mc_free(c->d_pah_W); mc_free(c->d_pah_P); mc_free(c->d_pah_J); mc_free(c->d_pah_next); mc_free(c->d_pah_q);
  mc_free(c->d_pah_cdf); mc_free(c->d_pah_cold); mc_free(c->d_pah_cnt); mc_free(c->d_pah_W32);
  c->d_pah_W32 = nullptr;
  c->d_kabs_eq = c->d_pah_C = c->d_pah_E = c->d_pah_T = c->d_pah_U = c->d_pah_Lam = c->d_pah_W = c->d_pah_P = nullptr;
  c->d_pah_J = nullptr; c->d_pah_next = nullptr; c->d_pah_q = c->d_pah_cdf = c->d_pah_cold = nullptr; c->d_pah_cnt = nullptr;
  c->pah = false;
}
static void free_observer(mcrt_ctx* c) {
  mc_free(c->obs.sed_mu); mc_free(c->obs.image);
  c->obs.sed_mu = c->obs.image = nullptr;
  c->obs.n_mu = c->obs.n_pix = 0;
}
static void free_sources(mcrt_ctx* c) {
  mc_free(c->d_src); mc_free(c->d_csrc); mc_free(c->d_csrc32);
  c->d_src = nullptr; c->d_csrc = nullptr; c->d_csrc32 = nullptr;
}

// Root delta tables of a swept grid: [12 N] = the tables with kLutRegion on every step that crosses a region
// boundary, followed by the plain tables; and plain | plain for the last sweep.
static mcrt_status build_region_tables(mcrt_ctx* ctx, const int* lut6N, const int shape[3]) {
  const int N = ctx->N;
  std::vector<int> marked(12 * (size_t)N), plain2(12 * (size_t)N);
  for (size_t i = 0; i < 6 * (size_t)N; ++i) { marked[i] = marked[6 * (size_t)N + i] = plain2[i] = plain2[6 * (size_t)N + i] = lut6N[i]; }
  for (int a = 0; a < 3; ++a)
    for (int i = 0; i < N; ++i) {
      if (i != N - 1 && (i + 1) % shape[a] == 0) marked[(size_t)(2 * a) * N + i] = kLutRegion;          // i -> i+1
      const int ir = N - 1 - i;
      if (ir != 0 && ir % shape[a] == 0) marked[(size_t)(2 * a + 1) * N + i] = kLutRegion;              // ir -> ir-1
    }
  if (!ctx->d_lut_marked) CU(mc_malloc(&ctx->d_lut_marked, sizeof(int) * marked.size()));
  if (!ctx->d_lut_plain2) CU(mc_malloc(&ctx->d_lut_plain2, sizeof(int) * plain2.size()));
  CU(cudaMemcpy(ctx->d_lut_marked, marked.data(), sizeof(int) * marked.size(), cudaMemcpyHostToDevice));
  CU(cudaMemcpy(ctx->d_lut_plain2, plain2.data(), sizeof(int) * plain2.size(), cudaMemcpyHostToDevice));
  for (int a = 0; a < 3; ++a) ctx->region_cells[a] = shape[a];
  return MCRT_OK;
}

// ---- storage order <-> the caller's slot order (R22) ---------------------------------------------
// root part through the root layout, sub-cells (contiguous behind it) copied; macro-cube grids: the
// caller's slots are the N^3 cells, stored cube by cube behind the macro array.
static bool needs_reorder(const mcrt_ctx* ctx) { return ctx->macro || ctx->lay.bricked; }

static mcrt_status store_to_api_u64(mcrt_ctx* ctx, const unsigned long long* store, unsigned long long* out, cudaStream_t st) {
  if (ctx->macro) {
    const long long nf3 = ctx->slots;
    k_store_to_ext<unsigned long long><<<(unsigned)((nf3 + 255) / 256), 256, 0, st>>>(store + ctx->store_n3, out, ctx->lay_fine, nf3);
    ctx->launches++;
    return MCRT_OK;
  }
  k_store_to_ext<unsigned long long><<<(unsigned)((ctx->n3 + 255) / 256), 256, 0, st>>>(store, out, ctx->lay, ctx->n3);
  ctx->launches++;
  if (ctx->slots > ctx->n3)
    CU(cudaMemcpyAsync(out + ctx->n3, store + ctx->store_n3, 8 * (size_t)(ctx->slots - ctx->n3), cudaMemcpyDeviceToDevice, st));
  return MCRT_OK;
}
static mcrt_status api_to_store_u64(mcrt_ctx* ctx, const unsigned long long* in, unsigned long long* store, cudaStream_t st) {
  if (ctx->macro) {
    const long long nf3 = ctx->slots;
    CU(cudaMemsetAsync(store, 0, 8 * (size_t)ctx->store_n3, st));
    k_ext_to_store_u64<<<(unsigned)((nf3 + 255) / 256), 256, 0, st>>>(in, store + ctx->store_n3, ctx->lay_fine, nf3);
    ctx->launches++;
    return MCRT_OK;
  }
  k_ext_to_store_u64<<<(unsigned)((ctx->n3 + 255) / 256), 256, 0, st>>>(in, store, ctx->lay, ctx->n3);
  ctx->launches++;
  if (ctx->slots > ctx->n3)
    CU(cudaMemcpyAsync(store + ctx->store_n3, in + ctx->n3, 8 * (size_t)(ctx->slots - ctx->n3), cudaMemcpyDeviceToDevice, st));
  return MCRT_OK;
}
static mcrt_status trow_to_api_T(mcrt_ctx* ctx, float* out, cudaStream_t st) {
  const float lnTmin = (float)std::log(ctx->Tmin), dlnT = (float)ctx->dlnT;
  if (ctx->macro) {
    const long long nf3 = ctx->slots;
    k_trow_to_T_u<<<(unsigned)((nf3 + 255) / 256), 256, 0, st>>>(ctx->d_trow + ctx->store_n3, out, ctx->lay_fine, nf3, lnTmin, dlnT);
    ctx->launches++;
    return MCRT_OK;
  }
  k_trow_to_T_u<<<(unsigned)((ctx->n3 + 255) / 256), 256, 0, st>>>(ctx->d_trow, out, ctx->lay, ctx->n3, lnTmin, dlnT);
  ctx->launches++;
  if (ctx->slots > ctx->n3) {                                // sub-cells: same order in storage and in the getter
    const long long ns = ctx->slots - ctx->n3;
    k_trow_to_T<<<(unsigned)((ns + 255) / 256), 256, 0, st>>>(ctx->d_trow + ctx->store_n3, out + ctx->n3, ns, lnTmin, dlnT);
    ctx->launches++;
  }
  return MCRT_OK;
}

// dynamic shared memory of the transport kernel: opacity float4[nb], SED u32[3 nb], emitted u32[nb], then at
// a 64-byte boundary the root delta tables int[6 N] (+ the subcube rows int[6][16] on two-level grids)
// what the next launch uses: the one-bit form only on request (it measured 3 % SLOWER than global gathers on
// the 64^3 sphere: the walk is bound by instruction issue, not by the gathers; profiles/r02_summary.md)
static int staging_mode(const mcrt_ctx* ctx) {
  if (ctx->dens_off == 1 || ctx->pah) return 0;              // (the PAH instances of the kernel gather from global memory)
  if (ctx->dens_mode == 2 && ctx->dens_off != 2) return 0;
  return ctx->dens_mode;
}
static size_t transport_smem_bytes(const mcrt_ctx* ctx, bool region = false) {
  const size_t n_lut = ctx->uni ? (region ? 12 : 6) * (size_t)ctx->N : (size_t)lut_sub_offset(ctx->N) + 6 * kSubStride;
  size_t b = ((32 * (size_t)ctx->nb + 63) & ~(size_t)63) + sizeof(int) * n_lut;
  if (staging_mode(ctx)) b = ((b + 127) & ~(size_t)127) + ctx->stage_bytes + 16;   // staged density + its mbarrier
  return b;
}

constexpr size_t kMaxSmemPerBlock = 227u << 10;              // B200: opt-in limit of dynamic shared memory

// One bit per cell for a single-level grid that holds only two distinct densities and whose bits fit into shared
// memory (mcrt_set_density_staging(2); measured slower than global gathers, so it is prepared only on request: the
// scan of the density array costs a device-to-host copy that mcrt_grid_create should not pay -- 0.8 of its 2.2 ms
// on the 64^3 sphere).
static mcrt_status prepare_density_bits(mcrt_ctx* ctx) {
  const size_t kStageMax = 40u << 10;
  if (ctx->dens_mode != 0 || !ctx->uni || ctx->d_bits || (size_t)(ctx->store_slots + 7) / 8 > kStageMax) return MCRT_OK;
  CU(cudaDeviceSynchronize());
  std::vector<float> h((size_t)ctx->store_slots);
  CU(cudaMemcpy(h.data(), ctx->d_rho, 4 * h.size(), cudaMemcpyDeviceToHost));
  float v0 = h[0], v1 = h[0];
  bool two = true, have1 = false;
  for (float v : h) {
    if (v == v0 || (have1 && v == v1)) continue;
    if (!have1) { v1 = v; have1 = true; continue; }
    two = false;
    break;
  }
  if (!two) return MCRT_OK;
  const size_t words = (((size_t)ctx->store_slots + 31) / 32 + 3) & ~(size_t)3;   // 16-byte units
  std::vector<uint32_t> bits(words, 0u);
  for (size_t i = 0; i < h.size(); ++i)
    if (have1 && h[i] == v1) bits[i >> 5] |= 1u << (i & 31);
  CU(mc_malloc(&ctx->d_bits, 4 * words));
  CU(cudaMemcpy(ctx->d_bits, bits.data(), 4 * words, cudaMemcpyHostToDevice));
  ctx->dens_mode = 2;
  ctx->stage_bytes = (unsigned)(4 * words);
  ctx->pal0 = v0; ctx->pal1 = v1;
  return MCRT_OK;
}

extern "C" {

mcrt_status mcrt_grid_create(const mcrt_grid_desc* d, mcrt_ctx** out) {
  mcrt_ctx* ctx = nullptr;
  if (!d || !out) return fail(nullptr, MCRT_EINVAL, "mcrt_grid_create: NULL argument");
  *out = nullptr;
  if (d->n_root < 1 || d->n_root > 1290 || !(d->root_size > 0) || !d->rho_root)
    return fail(nullptr, MCRT_EINVAL, "mcrt_grid_create: bad n_root / root_size / rho_root");
  if (d->sub < 0 || d->sub > 8) return fail(nullptr, MCRT_EINVAL, "mcrt_grid_create: sub must be 0..8");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(nullptr, MCRT_ECUDA, "mcrt_grid_create: no CUDA device (there is no CPU fallback)");
  ctx = new (std::nothrow) mcrt_ctx;
  if (!ctx) return fail(nullptr, MCRT_ENOMEM, "mcrt_grid_create: host allocation failed");
  struct Guard { mcrt_ctx* c; ~Guard() { if (c) mcrt_destroy(c); } } guard{ctx};
  auto bail = [&](mcrt_status st) { g_err = ctx->err; return st; };
#define CUG(call)                                                                         \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess)                                                                \
      return bail(fail(ctx, e_ == cudaErrorMemoryAllocation ? MCRT_ENOMEM : MCRT_ECUDA,   \
                       std::string(#call) + ": " + cudaGetErrorString(e_)));              \
  } while (0)
  CUG(cudaGetDevice(&ctx->device));
  int cc_major = 0;                                          // (attributes: cudaGetDeviceProperties costs ~1 ms)
  CUG(cudaDeviceGetAttribute(&cc_major, cudaDevAttrComputeCapabilityMajor, ctx->device));
  if (cc_major < 10)
    return bail(fail(ctx, MCRT_ECUDA, "mcrt_grid_create: device is not sm_100 class (built for sm_100a only)"));
  CUG(cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device));
  CUG(cudaDeviceGetAttribute(&ctx->coop_launch, cudaDevAttrCooperativeLaunch, ctx->device));
  ctx->N = d->n_root;
  ctx->S = d->sub > 1 ? d->sub : 1;
  ctx->root_size = d->root_size;
  for (int a = 0; a < 3; ++a) ctx->origin[a] = d->origin[a];
  const long long n3 = (long long)d->n_root * d->n_root * d->n_root;
  ctx->n3 = n3;
  // refined-cube numbering (k counts flagged cubes in x-fastest order)
  std::vector<int> refidx;
  long long k = 0;
  if (d->refine && ctx->S > 1) {
    std::vector<uint8_t> ref(n3);
    if (d->mem == MCRT_DEVICE) CUG(cudaMemcpy(ref.data(), d->refine, n3, cudaMemcpyDeviceToHost));
    else std::memcpy(ref.data(), d->refine, n3);
    refidx.assign(n3, -1);
    for (long long i = 0; i < n3; ++i) if (ref[i]) refidx[i] = (int)k++;
  }
  ctx->n_ref = k;
  if (k == 0) ctx->S = 1;
  const long long s3 = (long long)ctx->S * ctx->S * ctx->S;
  ctx->slots = n3 + k * s3;
  if (ctx->slots >= (1ll << 31)) return bail(fail(ctx, MCRT_EINVAL, "mcrt_grid_create: more than 2^31-1 leaf slots"));
  if (k > 0 && !d->rho_sub) return bail(fail(ctx, MCRT_EINVAL, "mcrt_grid_create: rho_sub is NULL but cubes are refined"));
  // storage order of the root grid (both kinds of grid; sub-cells always follow as blocks of S^3)
  if (d->layout < 0 || d->layout > 4) return bail(fail(ctx, MCRT_EINVAL, "mcrt_grid_create: layout must be 0..4"));
  ctx->uni = k == 0;
  ctx->lay.N = d->n_root;
  ctx->lay.nbk = (d->n_root + 7) / 8;
  // automatic: bricks for root grids larger than 48 MB -- single-level (c4) and, since the packages of a warp fly
  // closely together (64 x 128 start-direction bins), two-level ones too: c3 5.89 -> 5.72 ms per launch (it measured
  // slower before that, 13.3 vs 12.2 ms, when most of its gathers missed the L1 either way); c2 (12.8 MB) keeps
  // the x-fastest root (2.82 both ways)
  ctx->lay.bricked = d->layout == 2 || (d->layout == 0 && n3 * 4 > (48ll << 20));
  ctx->store_n3 = slots_of(ctx->lay);
  if (ctx->store_n3 + k * s3 >= (1ll << 31)) {               // padding pushed it over: fall back
    ctx->lay.bricked = 0;
    ctx->store_n3 = n3;
  }
  ctx->store_slots = ctx->store_n3 + k * s3;
  // staging copies of caller data (freed before returning)
  float *st_root = nullptr, *st_sub = nullptr;
  int* d_refidx = nullptr;
  const float *src_root = d->rho_root, *src_sub = d->rho_sub;
  struct Tmp { float*& a; float*& b; int*& c; ~Tmp() { mc_free(a); mc_free(b); mc_free(c); } } tmp{st_root, st_sub, d_refidx};
  if (d->mem == MCRT_HOST) {
    CUG(mc_malloc(&st_root, sizeof(float) * n3));
    CUG(cudaMemcpy(st_root, d->rho_root, sizeof(float) * n3, cudaMemcpyHostToDevice));
    src_root = st_root;
    if (k > 0) {
      CUG(mc_malloc(&st_sub, sizeof(float) * k * s3));
      CUG(cudaMemcpy(st_sub, d->rho_sub, sizeof(float) * k * s3, cudaMemcpyHostToDevice));
      src_sub = st_sub;
    }
  }
  // ---- macro cubes (on request: layout 3 / 4): a single-level grid run as a two-level one, 4^3 (8^3) blocks of
  // cells that hold ONE density are crossed in one step.  Not automatic any more: since the plain walk takes 35
  // instead of 42 instructions per crossing it is ahead on the 64^3 sphere for tau_V >= 1 (0.308 vs 0.316 ms per
  // 2^20 packages at tau_V = 1, 0.603 vs 0.627 at 100); the macro cubes still win where flights are long and
  // cross many uniform cubes (tau_V = 0.1: 0.212 vs 0.228 ms).  profiles/r02_summary.md
  if (k == 0 && d->layout >= 3) {
    const int M = d->layout == 4 ? 8 : 4;
    if (d->n_root % M == 0 && d->n_root / M >= 2 && n3 + n3 / (M * M * M) < (1ll << 31)) {
      const int Nm = d->n_root / M;
      const long long nm3 = (long long)Nm * Nm * Nm;
      {
        ctx->macro = M;
        ctx->n_fine = d->n_root;
        ctx->lay_fine.N = d->n_root; ctx->lay_fine.bricked = 2; ctx->lay_fine.nbk = Nm; ctx->lay_fine.bm = M;
        ctx->N = Nm; ctx->S = M; ctx->root_size = d->root_size * M;
        ctx->lay.N = Nm; ctx->lay.bricked = 0; ctx->lay.nbk = (Nm + 7) / 8;
        ctx->uni = false;                                      // the two-level kernel runs it
        ctx->n3 = nm3; ctx->store_n3 = nm3;
        ctx->store_slots = nm3 + n3;                           // macro array, then the cells cube by cube
        ctx->slots = n3;                                       // the caller's leaf slots stay the N^3 cells
      }
    }
  }
  CUG(mc_malloc(&ctx->d_rho, sizeof(float) * ctx->store_slots));
  CUG(mc_malloc(&ctx->d_tally, sizeof(unsigned long long) * ctx->store_slots));
  CUG(mc_malloc(&ctx->d_trow, sizeof(float) * ctx->store_slots));
  CUG(cudaMemset(ctx->d_tally, 0, sizeof(unsigned long long) * ctx->store_slots));
  CUG(cudaMemset(ctx->d_trow, 0, sizeof(float) * ctx->store_slots));
  if (k > 0) {
    CUG(mc_malloc(&d_refidx, sizeof(int) * n3));
    CUG(cudaMemcpy(d_refidx, refidx.data(), sizeof(int) * n3, cudaMemcpyHostToDevice));
  }
  {
    // per-axis slot-delta tables of the root grid: forward (i -> i+1) and reversed (entry j: i = N-1-j -> i-1);
    // two-level grids: followed by the tables of the S^3 subcubes of a refined cube (entry j = directional
    // subcube index: +-S^a, the last one = "leaves the cube")
    const int N = ctx->N, S = ctx->S;
    const size_t sub0 = (size_t)lut_sub_offset(N);
    std::vector<int> lut(ctx->uni ? 6 * (size_t)N : sub0 + 6 * kSubStride, 0);
    for (int a = 0; a < 3; ++a)
      for (int i = 0; i < N; ++i) {
        lut[(size_t)(2 * a) * N + i] = i == N - 1 ? kLutEscape
            : (int)(axis_term(ctx->lay, a, i + 1) - axis_term(ctx->lay, a, i));
        int ir = N - 1 - i;
        lut[(size_t)(2 * a + 1) * N + i] = ir == 0 ? kLutEscape
            : (int)(axis_term(ctx->lay, a, ir - 1) - axis_term(ctx->lay, a, ir));
      }
    if (!ctx->uni) {
      int stride = 1;
      for (int a = 0; a < 3; ++a) {
        for (int j = 0; j < S; ++j) {
          lut[sub0 + (size_t)(2 * a) * kSubStride + j] = j == S - 1 ? kLutLeave : stride;
          lut[sub0 + (size_t)(2 * a + 1) * kSubStride + j] = j == S - 1 ? kLutLeave : -stride;
        }
        lut[sub0 + (size_t)(2 * a) * kSubStride + kSubStride - 1] = -(S - 1) * stride;      // wrap to the mirror subcube
        lut[sub0 + (size_t)(2 * a + 1) * kSubStride + kSubStride - 1] = (S - 1) * stride;
        stride *= S;
      }
    }
    CUG(mc_malloc(&ctx->d_lut, sizeof(int) * lut.size()));
    CUG(cudaMemcpy(ctx->d_lut, lut.data(), sizeof(int) * lut.size(), cudaMemcpyHostToDevice));
    // Region sweeps for single-level bricked grids of at least 256^3 cells (the L2 and more): the root tables once
    // more with a marker on every step that crosses a boundary between regions of 256 x 128 x 128 cells (17 MB of
    // density: two of them in flight stay L2-resident; measured best on the 512^3 cube, profiles/r02_summary.md).
    constexpr int kRegionCells = 128;
    if (ctx->uni && ctx->lay.bricked == 1 && N >= 2 * kRegionCells && N % kRegionCells == 0) {
      const int shape[3] = {N % (2 * kRegionCells) == 0 && N >= 4 * kRegionCells ? 2 * kRegionCells : kRegionCells,
                            kRegionCells, kRegionCells};
      if (build_region_tables(ctx, lut.data(), shape) != MCRT_OK) return bail(MCRT_ECUDA);
    }
    CUG(cudaMemset(ctx->d_rho, 0, sizeof(float) * ctx->store_slots));
    if (ctx->macro) {
      // the cells cube by cube behind the macro array; then one entry per macro cube: its density if all
      // its cells hold the same one, else the marker (sign bit | slot of its first cell) that sends the walk to the cells
      k_encode_uniform<<<(unsigned)((n3 + 255) / 256), 256>>>(src_root, ctx->d_rho + ctx->store_n3, ctx->lay_fine, n3);
      k_macro_entries<<<(unsigned)((ctx->n3 + 127) / 128), 128>>>(ctx->d_rho + ctx->store_n3, ctx->d_rho, ctx->n3,
                                                                ctx->macro * ctx->macro * ctx->macro, ctx->store_n3);
      ctx->launches++;
    } else if (ctx->uni) k_encode_uniform<<<(unsigned)((n3 + 255) / 256), 256>>>(src_root, ctx->d_rho, ctx->lay, n3);
    else k_encode_root<<<(unsigned)((n3 + 255) / 256), 256>>>(src_root, d_refidx, ctx->d_rho, ctx->lay, n3, ctx->store_n3, (int)s3);
  }
  ctx->launches++;
  if (k > 0) {
    k_sanitize<<<(unsigned)((k * s3 + 255) / 256), 256>>>(src_sub, ctx->d_rho + ctx->store_n3, k * s3);
    ctx->launches++;
  }
  CUG(mc_malloc(&ctx->d_lnrho, sizeof(float) * ctx->store_slots));
  k_ln_density<<<(unsigned)((ctx->store_slots + 255) / 256), 256>>>(ctx->d_rho, ctx->d_lnrho, ctx->store_slots);
  ctx->launches++;
  CUG(cudaGetLastError());
  CUG(cudaDeviceSynchronize());
  // Small single-level problems keep their density in shared memory (transport_u.cuh, DENS): the array itself
  // if it is at most 40 KB, or one bit per slot if it holds only two distinct values and the bits fit.
  if (ctx->uni) {
    const size_t kStageMax = 40u << 10;
    if ((size_t)ctx->store_slots * 4 <= kStageMax) {
      ctx->dens_mode = 1;
      ctx->stage_bytes = (unsigned)(((size_t)ctx->store_slots * 4 + 15) & ~(size_t)15);
      if (ctx->stage_bytes > (size_t)ctx->store_slots * 4) {   // the bulk copy reads whole 16-byte units
        float* padded = nullptr;
        CUG(mc_malloc(&padded, ctx->stage_bytes));
        CUG(cudaMemset(padded, 0, ctx->stage_bytes));
        CUG(cudaMemcpy(padded, ctx->d_rho, (size_t)ctx->store_slots * 4, cudaMemcpyDeviceToDevice));
        mc_free(ctx->d_rho);
        ctx->d_rho = padded;
      }
    }
  }
  guard.c = nullptr;
  *out = ctx;
  return MCRT_OK;
#undef CUG
}

mcrt_status mcrt_destroy(mcrt_ctx* ctx) {
  if (!ctx) return MCRT_EINVAL;
  DeviceScope scope(ctx->device);                            // the context's GPU, whichever is current in the caller
  cudaDeviceSynchronize();                                   // nothing of this context may still be running
  DeviceIdleScope idle;                                      // ... and nothing is launched below: the frees need not wait again
  for (auto& b : ctx->pending) { cudaEventDestroy(b.e0); cudaEventDestroy(b.e1); cudaEventDestroy(b.e2); }
  for (auto& b : ctx->spare) { cudaEventDestroy(b.e0); cudaEventDestroy(b.e1); cudaEventDestroy(b.e2); }
  for (auto& t : ctx->tickets) {
    mc_free(t.snap_abs); mc_free(t.snap_T); mc_free(t.snap_small); cudaFreeHost(t.h_small);
    if (t.ev_snap) cudaEventDestroy(t.ev_snap);
    if (t.ev_done) cudaEventDestroy(t.ev_done);
  }
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  free_opacity(ctx);
  free_pah(ctx);
  free_sources(ctx);
  free_observer(ctx);
  mc_free(ctx->d_rho); mc_free(ctx->d_lnrho); mc_free(ctx->d_tally); mc_free(ctx->d_trow);
  mc_free(ctx->d_lut); mc_free(ctx->d_lut_marked); mc_free(ctx->d_lut_plain2); mc_free(ctx->d_rec);
  mc_free(ctx->d_list[0]); mc_free(ctx->d_list[1]); mc_free(ctx->d_swcnt); mc_free(ctx->d_regcnt);
  mc_free(ctx->d_heads);
  mc_free(ctx->d_bits); mc_free(ctx->d_tally_scratch); mc_free(ctx->d_perm); mc_free(ctx->d_keys); mc_free(ctx->d_srccnt); mc_free(ctx->d_out_scratch);
  delete ctx;
  return MCRT_OK;
}

int64_t mcrt_leaf_slots(const mcrt_ctx* ctx) { return ctx ? ctx->slots : -1; }

mcrt_status mcrt_set_opacity(mcrt_ctx* ctx, const mcrt_opacity_desc* d) {
  if (!ctx) return MCRT_EINVAL;
  if (!d || !d->lambda_edges_um || !d->weight || !d->kabs || !d->ksca || !d->g)
    return fail(ctx, MCRT_EINVAL, "mcrt_set_opacity: NULL argument");
  if (d->n_bins < 1 || d->n_bins > 4096 || d->n_species < 1)
    return fail(ctx, MCRT_EINVAL, "mcrt_set_opacity: n_bins must be 1..4096, n_species >= 1");
  for (int j = 0; j < d->n_bins; ++j)
    if (!(d->lambda_edges_um[j] > 0) || !(d->lambda_edges_um[j + 1] > d->lambda_edges_um[j]))
      return fail(ctx, MCRT_EINVAL, "mcrt_set_opacity: wavelength edges must be positive and ascending");
  {
    mcrt_ctx probe;                                          // same formula as the launch, with the new n_bins
    probe.nb = d->n_bins; probe.N = ctx->N; probe.uni = ctx->uni;
    if (transport_smem_bytes(&probe) > kMaxSmemPerBlock)
      return fail(ctx, MCRT_EINVAL, "mcrt_set_opacity: 32*n_bins + 24*n_root bytes of shared memory per block exceed 227 KB");
  }
  int nT = d->n_T;
  double Tmin = d->T_min, Tmax = d->T_max;
  if (nT == 0) { nT = 801; Tmin = 1.0; Tmax = 1.0e4; }
  if (nT < 2 || nT > 8192 || !(Tmin > 0) || !(Tmax > Tmin))
    return fail(ctx, MCRT_EINVAL, "mcrt_set_opacity: bad temperature table");
  for (auto& t : ctx->tickets)
    if (t.busy) return fail(ctx, MCRT_ESTATE, "mcrt_set_opacity: a read-out ticket is in flight (call mcrt_results_wait first)");
  CU(cudaDeviceSynchronize());
  for (auto& t : ctx->tickets) { mc_free(t.snap_small); t.snap_small = nullptr; }   // sized by n_bins
  free_opacity(ctx);
  free_pah(ctx);                                            // a PAH is declared against an opacity set
  free_sources(ctx);
  free_observer(ctx);                                       // its tallies are sized by n_bins
  ctx->have_opacity = ctx->have_source = false;
  const int nb = d->n_bins, ns = d->n_species;
  ctx->nb = nb; ctx->nT = nT; ctx->Tmin = Tmin; ctx->Tmax = Tmax;
  ctx->dlnT = (std::log(Tmax) - std::log(Tmin)) / (nT - 1);
  double *d_edges = nullptr, *d_w = nullptr;
  float *d_ka = nullptr, *d_ks = nullptr, *d_g = nullptr;
  struct Tmp { double*& a; double*& b; float*& c; float*& d; float*& e;
               ~Tmp() { mc_free(a); mc_free(b); mc_free(c); mc_free(d); mc_free(e); } } tmp{d_edges, d_w, d_ka, d_ks, d_g};
  CU(mc_malloc(&d_edges, 8 * (nb + 1))); CU(mc_malloc(&d_w, 8 * ns));
  CU(mc_malloc(&d_ka, 4 * (size_t)ns * nb)); CU(mc_malloc(&d_ks, 4 * (size_t)ns * nb));
  CU(mc_malloc(&d_g, 4 * (size_t)ns * nb));
  CU(cudaMemcpy(d_edges, d->lambda_edges_um, 8 * (nb + 1), cudaMemcpyHostToDevice));
  CU(cudaMemcpy(d_w, d->weight, 8 * ns, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(d_ka, d->kabs, 4 * (size_t)ns * nb, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(d_ks, d->ksca, 4 * (size_t)ns * nb, cudaMemcpyHostToDevice));
  CU(cudaMemcpy(d_g, d->g, 4 * (size_t)ns * nb, cudaMemcpyHostToDevice));
  CU(mc_malloc(&ctx->d_nu, 8 * nb)); CU(mc_malloc(&ctx->d_dnu, 8 * nb)); CU(mc_malloc(&ctx->d_kabs, 8 * nb));
  CU(mc_malloc(&ctx->d_opac, sizeof(float4) * nb));
  CU(mc_malloc(&ctx->d_lnQ, 4 * nT));
  CU(mc_malloc(&ctx->d_cdf, 4 * (size_t)nT * nb));
  CU(mc_malloc(&ctx->d_guide, sizeof(int) * kGuide));
  CU(mc_malloc(&ctx->d_cdf_guide, sizeof(uint32_t) * (size_t)nT * kCdfGuide));
  const size_t n_small = 1 + CNT_N + 4 * (size_t)nb;
  CU(mc_malloc(&ctx->d_small, 8 * n_small));
  CU(cudaMemset(ctx->d_small, 0, 8 * n_small));
  k_mix_opacity<<<(nb + 127) / 128, 128>>>(nb, ns, d_edges, d_w, d_ka, d_ks, d_g, ctx->root_size,
                                           ctx->d_nu, ctx->d_dnu, ctx->d_kabs, ctx->d_opac);
  k_build_emission_rows<<<nT, 128, 8 * (nb + 1)>>>(nb, nT, Tmin, Tmax, ctx->d_nu, ctx->d_dnu,
                                                   ctx->d_kabs, ctx->d_lnQ, ctx->d_cdf);
  k_build_guide<<<kGuide / 256, 256>>>(ctx->d_lnQ, nT, ctx->d_guide);
  k_build_cdf_guide<<<nT, kCdfGuide>>>(ctx->d_cdf, nb, nT, ctx->d_cdf_guide);
  ctx->launches += 4;
  CU(cudaGetLastError());
  CU(cudaDeviceSynchronize());
  ctx->have_opacity = true;
  return MCRT_OK;
}

mcrt_status mcrt_set_source(mcrt_ctx* ctx, int32_t n_src, const mcrt_source* src) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_set_source: call mcrt_set_opacity first");
  if (n_src < 1 || n_src > 65536 || !src) return fail(ctx, MCRT_EINVAL, "mcrt_set_source: bad n_src / NULL");
  std::vector<SrcDev> h(n_src);
  std::vector<double> Tbb(n_src);
  double Ltot = 0;
  for (int s = 0; s < n_src; ++s) {
    if (!(src[s].L > 0) || !(src[s].T_bb > 0) || (src[s].type != 0 && src[s].type != 1))
      return fail(ctx, MCRT_EINVAL, "mcrt_set_source: L and T_bb must be > 0, type 0 or 1");
    Ltot += src[s].L;
  }
  double acc = 0;
  const int Sf = ctx->S;
  for (int s = 0; s < n_src; ++s) {
    h[s].type = src[s].type;
    Tbb[s] = src[s].T_bb;
    acc += src[s].L;
    h[s].lcdf = s == n_src - 1 ? 1.0 : acc / Ltot;
    for (int a = 0; a < 3; ++a) { h[s].fine[a] = 0; h[s].frac[a] = 0.f; }
    if (src[s].type == 0) {
      for (int a = 0; a < 3; ++a) {
        double xf = (src[s].pos[a] - ctx->origin[a]) / ctx->root_size * Sf;   // finest-level units
        if (!(xf > 0.0) || !(xf < (double)ctx->N * Sf))
          return fail(ctx, MCRT_EINVAL, "mcrt_set_source: point source outside the grid");
        double fl = std::floor(xf);
        float fr = (float)(xf - fl);
        if (fr >= 1.f) { fl += 1.0; fr = 0.f; }             // the fraction rounded up to the next cell
        if (fl >= (double)ctx->N * Sf)                       // ... which must still lie inside the grid
          return fail(ctx, MCRT_EINVAL, "mcrt_set_source: point source outside the grid");
        h[s].fine[a] = (int)fl;
        h[s].frac[a] = fr;
      }
    }
  }
  CU(cudaDeviceSynchronize());
  free_sources(ctx);
  ctx->have_source = false;
  double* d_T = nullptr;
  struct Tmp { double*& a; ~Tmp() { mc_free(a); } } tmp{d_T};
  CU(mc_malloc(&d_T, 8 * n_src));
  CU(cudaMemcpy(d_T, Tbb.data(), 8 * n_src, cudaMemcpyHostToDevice));
  CU(mc_malloc(&ctx->d_src, sizeof(SrcDev) * n_src));
  CU(cudaMemcpy(ctx->d_src, h.data(), sizeof(SrcDev) * n_src, cudaMemcpyHostToDevice));
  CU(mc_malloc(&ctx->d_csrc, 8 * (size_t)n_src * ctx->nb));
  CU(mc_malloc(&ctx->d_csrc32, 4 * (size_t)n_src * ctx->nb));
  k_build_source_cdf<<<n_src, 128, 8 * (ctx->nb + 1)>>>(ctx->nb, d_T, ctx->d_nu, ctx->d_dnu, ctx->d_csrc, ctx->d_csrc32);
  ctx->launches++;
  CU(cudaGetLastError());
  CU(cudaDeviceSynchronize());
  ctx->nsrc = n_src;
  ctx->Ltot = Ltot;
  ctx->have_source = true;
  return MCRT_OK;
}

static mcrt_status take_events(mcrt_ctx* ctx, BatchEvents* b) {
  if (!ctx->spare.empty()) { *b = ctx->spare.back(); ctx->spare.pop_back(); return MCRT_OK; }
  CU(cudaEventCreate(&b->e0)); CU(cudaEventCreate(&b->e1)); CU(cudaEventCreate(&b->e2));
  return MCRT_OK;
}

// tally32 != NULL (packet-sharded batch): uint32[store slots] for the equilibrium grains, followed -- when a PAH is
// declared -- by uint32[store slots][n_bins] for the PAH's absorbed spectrum; this batch's counts only.
// fused != NULL: the caller wants the temperature update (a9) of THIS batch (n_cum = ctx->Ncum + n) at the end of the
// same launch; *fused says whether that was done (one cooperative launch; not on swept grids, with a PAH, for
// sharded batches or when the device cannot launch cooperatively -- then the caller launches k_update_temperature).
static mcrt_status launch_transport(mcrt_ctx* ctx, uint64_t seed, uint64_t first, uint64_t n, cudaStream_t st,
                                    uint32_t* tally32 = nullptr, bool* fused = nullptr) {
  if (fused) *fused = false;
  if (n == 0) return MCRT_OK;
  const uint64_t kMaxLaunch = 1ull << 31;                    // the kernels number packages within a launch in 32 bits
  if (n > kMaxLaunch) {
    mcrt_status rc = launch_transport(ctx, seed, first, kMaxLaunch, st, tally32);
    if (rc != MCRT_OK) return rc;
    return launch_transport(ctx, seed, first + kMaxLaunch, n - kMaxLaunch, st, tally32);
  }
  const int nb = ctx->nb;
  TransportParams P;
  P.rho = ctx->d_rho; P.tally = ctx->d_tally; P.tally32 = tally32; P.trow = ctx->d_trow;
  P.cdf_guide = ctx->cdf_guide_off ? nullptr : ctx->d_cdf_guide;
  P.opac = ctx->d_opac; P.cdf = ctx->d_cdf; P.csrc = ctx->d_csrc32; P.csrc64 = ctx->d_csrc; P.src = ctx->d_src;
  if (!ctx->d_heads) {
    CU(mc_malloc(&ctx->d_heads, 16));
    CU(cudaMemset(ctx->d_heads, 0, 16));
  }
  P.next = nullptr; P.next_reset = nullptr;                  // (set at each launch, below)
  P.counters = ctx->d_small + 1;
  P.sed = ctx->d_small + 1 + CNT_N; P.emit_bin = P.sed + 3 * (size_t)nb;
  P.seed = seed; P.first = first; P.count = n;
  P.obs = ctx->obs;
  P.pah_q = ctx->pah ? ctx->d_pah_q : nullptr; P.pah_cdf = ctx->d_pah_cdf;
  P.pah_cnt = (ctx->pah && tally32) ? tally32 + ctx->store_slots : ctx->d_pah_cnt;
  P.N = ctx->N; P.S = ctx->S; P.nb = nb; P.nT = ctx->nT; P.nsrc = ctx->nsrc; P.n3 = (int)ctx->store_n3;
#ifdef MCRT_CHECKS
  CU(cudaMemcpyToSymbolAsync(g_mcrt_nstore, &ctx->store_slots, sizeof(long long), 0, cudaMemcpyHostToDevice, st));
#endif
  P.perm = nullptr;
  const bool big = (size_t)ctx->store_slots * 4 > ((size_t)48 << 20);
  // 0 off, 1 grouped by source, 2 by source and start direction; automatic: 2 when the pre-pass is
  // small against the batch (grid larger than the L2, or at least 2^21 packages)
  int gmode = ctx->order_by_source < 0 ? ((big || n >= (1ull << 21)) ? 2 : 0) : ctx->order_by_source;
  if (gmode == 1 && ctx->nsrc < 2) gmode = 0;
  int sub = 1;                                               // start-direction sub-groups per source
  if (gmode == 2) {                                          // the finest direction bins the group table has room for
    sub = 1;
    for (int m = 64; m >= 4 && sub == 1; m >>= 1)            // ... and the batch has packages for (256 per group on average)
      if ((long long)ctx->nsrc * 2 * m * m <= kMaxOrderedSources && ((long long)ctx->nsrc * 2 * m * m * 256 <= (long long)n || m == 4))
        sub = 2 * m * m;
  }
  if (gmode && sub * ctx->nsrc <= kMaxOrderedSources && (sub > 1 || ctx->nsrc > 1) && n >= 65536) {
    if (ctx->perm_cap < n) {
      mc_free(ctx->d_perm); ctx->d_perm = nullptr; ctx->perm_cap = 0;
      CU(mc_malloc(&ctx->d_perm, sizeof(uint32_t) * (size_t)n));
      ctx->perm_cap = n;
    }
    if (ctx->keys_cap < n) {
      mc_free(ctx->d_keys); ctx->d_keys = nullptr; ctx->keys_cap = 0;
      CU(mc_malloc(&ctx->d_keys, sizeof(uint16_t) * (size_t)n));
      ctx->keys_cap = n;
    }
    if (!ctx->d_srccnt) CU(mc_malloc(&ctx->d_srccnt, sizeof(unsigned int) * 2 * kMaxOrderedSources));
    CU(cudaMemsetAsync(ctx->d_srccnt, 0, sizeof(unsigned int) * 2 * kMaxOrderedSources, st));
    // (every block flushes its histogram of all groups: fewer, larger blocks when the groups are many)
    const unsigned gblocks = (unsigned)ctx->sm_count * (ctx->nsrc * sub > 2048 ? 3u : 8u);
    const size_t gsmem = sizeof(unsigned int) * 2 * (size_t)ctx->nsrc * sub;
    if (gsmem > (48u << 10) && !ctx->group_smem_set) {
      CU(cudaFuncSetAttribute(k_group_by_source, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(sizeof(unsigned int) * 2 * kMaxOrderedSources)));
      ctx->group_smem_set = true;
    }
    k_group_by_source<<<gblocks, 256, gsmem, st>>>(P, sub, ctx->d_srccnt, nullptr, nullptr, ctx->d_keys);
    k_scan_sources<<<1, 1024, 0, st>>>(ctx->d_srccnt, ctx->d_srccnt + kMaxOrderedSources, ctx->nsrc * sub);
    k_group_by_source<<<gblocks, 256, gsmem, st>>>(P, sub, ctx->d_srccnt, ctx->d_srccnt + kMaxOrderedSources, ctx->d_perm, ctx->d_keys);
    ctx->launches += 3;
    P.perm = ctx->d_perm;
  }
  const int threads = ctx->threads;
  // resident blocks per SM: the caller's choice, else 5 (48-register kernels), except 4 for the
  // single-level kernel on HBM-resident grids (bricked storage), where more threads thrash the L1
  // (and 4 for macro-cube grids: the 48-register build of that instance spills in the walk, c1_tau1 0.337 vs 0.329 ms)
  const int bps = ctx->blocks_per_sm ? ctx->blocks_per_sm : ((ctx->uni && ctx->lay.bricked) || ctx->macro ? 4 : 5);
  long long want = ((long long)n + threads - 1) / threads;
  long long grid = (long long)ctx->sm_count * bps;
  if (want < grid) grid = want;
  // region sweeps: automatic for qualifying grids and batches of at least 2^20 packages
  constexpr int kMaxSweeps = 30;
  int sweeps = 0;
  if (ctx->region_cells[0] && !ctx->pah) {                   // (either tally; the PAH split is not carried in a record)
    if (ctx->region_sweeps < 0) sweeps = n >= (1ull << 20) ? 6 : 0;          // automatic
    else sweeps = ctx->region_sweeps > kMaxSweeps ? kMaxSweeps : ctx->region_sweeps;   // forced: any batch size
  }
  const bool region = sweeps > 0;
  const size_t smem = transport_smem_bytes(ctx, region);
  TransportParamsU PU;
  const int tail_mode = ctx->tail_mode < 0 ? 3 : ctx->tail_mode;
  PU.tail = tail_mode & 1;
  PU.base = P; PU.lut = ctx->d_lut; PU.lay = ctx->lay; PU.quorum = ctx->quorum;
  PU.rec = nullptr; PU.list_out = nullptr; PU.list_out_count = nullptr; PU.count_dev = nullptr; PU.resume = 0;
  for (int a = 0; a < 3; ++a) {
    PU.region_cells[a] = ctx->region_cells[a] ? ctx->region_cells[a] : 1;
    PU.regions_per_axis[a] = ctx->region_cells[a] ? ctx->N / ctx->region_cells[a] : 1;
  }
  PU.lut2 = 0;
  if (region) {
    if (ctx->rec_cap < n) {
      mc_free(ctx->d_rec); mc_free(ctx->d_list[0]); mc_free(ctx->d_list[1]);
      ctx->d_rec = nullptr; ctx->d_list[0] = ctx->d_list[1] = nullptr; ctx->rec_cap = 0;
      CU(mc_malloc(&ctx->d_rec, sizeof(float4) * 3 * (size_t)n));
      CU(mc_malloc(&ctx->d_list[0], 8 * (size_t)n));
      CU(mc_malloc(&ctx->d_list[1], 8 * (size_t)n));
      ctx->rec_cap = n;
    }
    if (ctx->perm_cap < n) {
      mc_free(ctx->d_perm); ctx->d_perm = nullptr; ctx->perm_cap = 0;
      CU(mc_malloc(&ctx->d_perm, sizeof(uint32_t) * (size_t)n));
      ctx->perm_cap = n;
    }
    const int nreg = 4096;                                   // capacity of the histogram (regions <= 4096)
    if (!ctx->d_swcnt) CU(mc_malloc(&ctx->d_swcnt, sizeof(unsigned int) * (kMaxSweeps + 2)));
    if (!ctx->d_regcnt) CU(mc_malloc(&ctx->d_regcnt, sizeof(unsigned int) * 2 * (size_t)nreg));
    CU(cudaMemsetAsync(ctx->d_swcnt, 0, sizeof(unsigned int) * (kMaxSweeps + 2), st));
    PU.rec = ctx->d_rec; PU.lut = ctx->d_lut_marked;
    PU.list_out = ctx->d_list[0]; PU.list_out_count = ctx->d_swcnt;
  }
  const int dens = staging_mode(ctx);
  PU.stage = dens == 1 ? (const void*)ctx->d_rho : (const void*)ctx->d_bits;
  PU.stage_bytes = ctx->stage_bytes; PU.pal0 = ctx->pal0; PU.pal1 = ctx->pal1;
  const bool five = bps * threads > 1024 && !ctx->pah;      // 48-register build (5 blocks of 256) or 64-register build
  void (*kern)(TransportParamsU) =
      ctx->pah ? (ctx->macro ? k_transport_u<4, true, 0, true, true, false>       // PAH instances: 64-register builds,
                  : !ctx->uni ? k_transport_u<4, true, 0, false, true, false>     // global gathers
                              : k_transport_u<4, false, 0, false, true, false>)
      : ctx->macro ? (five ? k_transport_u<5, true, 0, true, false, false> : k_transport_u<4, true, 0, true, false, false>)
      : !ctx->uni ? (five ? k_transport_u<5, true, 0, false, false, false> : k_transport_u<4, true, 0, false, false, false>)
      : region ? k_transport_u<4, false, 0, false, false, true>
      : dens == 1 ? k_transport_u<5, false, 1, false, false, false>
      : dens == 2 ? k_transport_u<5, false, 2, false, false, false>
                  : (five ? k_transport_u<5, false, 0, false, false, false> : k_transport_u<4, false, 0, false, false, false>);
  int resident = ctx->occ_resident;                          // large tables (many bins) lower the residency:
  if (ctx->occ_kern != (const void*)kern || ctx->occ_threads != threads || ctx->occ_smem != smem) {
    if (smem > (48u << 10)) CU(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (dens) CU(cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&resident, kern, threads, smem));   // size the grid to what fits
    ctx->occ_kern = (const void*)kern; ctx->occ_threads = threads; ctx->occ_smem = smem; ctx->occ_resident = resident;
  }
  if (resident < 1) return fail(ctx, MCRT_EINVAL, "mcrt_run_batch: the transport kernel does not fit on an SM with these tables");
  if ((long long)ctx->sm_count * resident < grid) grid = (long long)ctx->sm_count * resident;
  PU.base.next = ctx->d_heads + ctx->head; PU.base.next_reset = ctx->d_heads + (ctx->head ^ 1);
  ctx->head ^= 1;
  PU.upd_nT = 0;
  // (it pays on small grids only: C0's 10^4-package batches 0.052 -> 0.048 ms per step; at 2.7e5 leaves (C1) the
  // barrier and the update inside the kernel cost what the second launch did, from 3e6 leaves on (C2, C3) more: the
  // kernel of its own reads the tables from shared memory and two leaves per thread)
  constexpr long long kFuseUpdateMaxSlots = 65536;
  if (fused && !region && !ctx->pah && !tally32 && (tail_mode & 2) && ctx->coop_launch &&
      (ctx->store_slots <= kFuseUpdateMaxSlots || ctx->tail_mode == 2 || ctx->tail_mode == 3)) {
    const double PI = 3.14159265358979323846;
    const double V = ctx->root_size * ctx->root_size * ctx->root_size;
    PU.upd_nT = ctx->nT;
    PU.upd_ln_coef = (float)(std::log(ctx->Ltot) - std::log((double)(ctx->Ncum + n)) - std::log(4.0 * PI) - std::log(V));
    PU.upd_ln_sub3 = (float)(3.0 * std::log((double)ctx->S));
    PU.upd_lnQ = ctx->d_lnQ; PU.upd_guide = ctx->d_guide; PU.upd_trow = ctx->d_trow; PU.upd_lnrho = ctx->d_lnrho;
    PU.upd_slots = ctx->store_slots; PU.upd_n3 = ctx->uni ? ctx->store_slots : ctx->store_n3;
    void* args[] = {(void*)&PU};
    const cudaError_t ce = cudaLaunchCooperativeKernel((const void*)kern, dim3((unsigned)grid), dim3((unsigned)threads), args, smem, st);
    if (ce == cudaSuccess) {
      *fused = true;
    } else {                                                 // (e.g. the grid cannot be co-resident right now): two launches
      (void)cudaGetLastError();
      PU.upd_nT = 0;
      kern<<<(unsigned)grid, threads, smem, st>>>(PU);
    }
  } else {
    kern<<<(unsigned)grid, threads, smem, st>>>(PU);
  }
  ctx->launches++;
  CU(cudaGetLastError());
  if (region) {
    // sweeps 1..sweeps: the packages suspended in the previous sweep, grouped by the region they wait in; the last
    // one runs on plain tables (no markers) and finishes every package that is left
    const int nreg = PU.regions_per_axis[0] * PU.regions_per_axis[1] * PU.regions_per_axis[2];
    const long long full = (long long)ctx->sm_count * resident < (long long)ctx->sm_count * bps
                               ? (long long)ctx->sm_count * resident : (long long)ctx->sm_count * bps;
    for (int sw = 1; sw <= sweeps; ++sw) {
      const unsigned long long* list_in = ctx->d_list[(sw - 1) & 1];
      const unsigned int* n_in = ctx->d_swcnt + (sw - 1);
      CU(cudaMemsetAsync(ctx->d_regcnt, 0, sizeof(unsigned int) * 2 * (size_t)nreg, st));
      const unsigned gblocks = (unsigned)ctx->sm_count * 4u;
      k_region_hist<<<gblocks, 256, sizeof(unsigned int) * nreg, st>>>(list_in, n_in, nreg, ctx->d_regcnt);
      k_scan_sources<<<1, 1024, 0, st>>>(ctx->d_regcnt, ctx->d_regcnt + nreg, nreg);
      k_region_scatter<<<gblocks, 256, sizeof(unsigned int) * 2 * nreg, st>>>(list_in, n_in, nreg, ctx->d_regcnt + nreg, ctx->d_perm);
      PU.base.next = ctx->d_heads + ctx->head; PU.base.next_reset = ctx->d_heads + (ctx->head ^ 1);
      ctx->head ^= 1;
      PU.base.perm = ctx->d_perm;
      PU.resume = 1; PU.count_dev = n_in;
      PU.lut = sw == sweeps ? ctx->d_lut_plain2 : ctx->d_lut_marked;
      PU.list_out = ctx->d_list[sw & 1]; PU.list_out_count = ctx->d_swcnt + sw;
      kern<<<(unsigned)full, threads, smem, st>>>(PU);
      ctx->launches += 4;
      CU(cudaGetLastError());
    }
  }
  return MCRT_OK;
}

// a9 for the PAH (pah.cuh): P(T) and emission CDF of every leaf from its absorbed spectrum
static size_t pah_smem_bytes(const mcrt_ctx* ctx, int warps) {
  return sizeof(double) * (size_t)warps * (size_t)pah_warp_doubles(ctx->nb, ctx->pahd.K);
}
static mcrt_status launch_pah_update(mcrt_ctx* ctx, uint64_t n_cum, cudaStream_t st, long long only_slot) {
  if (n_cum == 0) return MCRT_OK;
  int warps = 4;
  while (warps > 1 && pah_smem_bytes(ctx, warps) > (96u << 10)) warps >>= 1;
  const size_t smem = pah_smem_bytes(ctx, warps);
  if (smem > (48u << 10)) CU(cudaFuncSetAttribute(k_pah_update, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  const double V = ctx->root_size * ctx->root_size * ctx->root_size;
  const double s3 = (double)ctx->S * ctx->S * ctx->S;
  long long blocks = only_slot >= 0 ? 1 : (ctx->store_slots + warps - 1) / warps;
  const long long cap = (long long)ctx->sm_count * 16;
  if (blocks > cap) blocks = cap;
  if (!ctx->d_pah_next) CU(mc_malloc(&ctx->d_pah_next, 8));
  CU(cudaMemsetAsync(ctx->d_pah_next, 0, 8, st));            // work queue of leaves
  k_pah_update<<<(unsigned)blocks, 32 * (only_slot >= 0 ? 1 : warps), smem, st>>>(
      ctx->pahd, ctx->d_rho, ctx->d_pah_cnt, ctx->d_pah_cdf, ctx->store_slots,
      ctx->uni ? ctx->store_slots : ctx->store_n3, ctx->Ltot / (double)n_cum, V, 1.0 / s3, only_slot, ctx->d_pah_P,
      ctx->d_pah_next);
  ctx->launches++;
  CU(cudaGetLastError());
  return MCRT_OK;
}

// a9: T from `tally` (the context's own cumulative tally, or a caller's device array that
// holds the sum over ranks) and n_cum packages emitted so far in the whole job.
// delta != NULL: first add the batch's counts (u32, storage order, summed over ranks) to the context's tally.
static mcrt_status launch_update(mcrt_ctx* ctx, const unsigned long long* tally, uint64_t n_cum, cudaStream_t st,
                                 const uint32_t* delta = nullptr) {
  if (n_cum == 0) return MCRT_OK;
  const double PI = 3.14159265358979323846;
  double V = ctx->root_size * ctx->root_size * ctx->root_size;
  float ln_coef = (float)(std::log(ctx->Ltot) - std::log((double)n_cum) - std::log(4.0 * PI) - std::log(V));
  float ln_sub3 = (float)(3.0 * std::log((double)ctx->S));
  if (tally != ctx->d_tally && needs_reorder(ctx)) {               // caller's sum is in slot order (R22)
    if (!ctx->d_tally_scratch) {
      CU(mc_malloc(&ctx->d_tally_scratch, 8 * (size_t)ctx->store_slots));
      CU(cudaMemsetAsync(ctx->d_tally_scratch, 0, 8 * (size_t)ctx->store_slots, st));
    }
    mcrt_status rc = api_to_store_u64(ctx, tally, ctx->d_tally_scratch, st);
    if (rc != MCRT_OK) return rc;
    tally = ctx->d_tally_scratch;
  }
  long long blocks = (ctx->store_slots / 2 + 256) / 256;     // two leaves per thread and turn
  long long cap = (long long)ctx->sm_count * 8;
  if (blocks > cap) blocks = cap;
  const size_t smem = 4 * (size_t)ctx->nT + sizeof(int) * kGuide;
  const long long n3 = ctx->uni ? ctx->store_slots : ctx->store_n3;
  if (delta)
    k_update_temperature<true><<<(unsigned)blocks, 256, smem, st>>>(ctx->d_lnrho, ctx->d_tally, delta, ctx->d_trow, ctx->d_lnQ,
                                                                    ctx->d_guide, ctx->nT, ctx->store_slots, n3, ln_coef, ln_sub3);
  else
    k_update_temperature<false><<<(unsigned)blocks, 256, smem, st>>>(ctx->d_lnrho, const_cast<unsigned long long*>(tally), nullptr,
                                                                     ctx->d_trow, ctx->d_lnQ, ctx->d_guide, ctx->nT,
                                                                     ctx->store_slots, n3, ln_coef, ln_sub3);
  ctx->launches++;
  CU(cudaGetLastError());
  if (ctx->pah) return launch_pah_update(ctx, n_cum, st, -1);
  return MCRT_OK;
}

static mcrt_status begin_batch(mcrt_ctx* ctx, BatchEvents* ev) {
  if (ctx->pending.size() >= 4096) {                         // nobody is reading the timings: recycle
    CU(cudaEventSynchronize(ctx->pending.back().e2));
    for (auto& b : ctx->pending) ctx->spare.push_back(b);
    ctx->pending.clear();
  }
  return take_events(ctx, ev);
}

mcrt_status mcrt_run_batch(mcrt_ctx* ctx, uint64_t seed, uint64_t first, uint64_t n, void* stream_) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->have_source) return fail(ctx, MCRT_ESTATE, "mcrt_run_batch: grid, opacity and sources must be set first");
  cudaStream_t st = (cudaStream_t)stream_;
  BatchEvents ev;
  mcrt_status rc = begin_batch(ctx, &ev);
  if (rc != MCRT_OK) return rc;
  CU(cudaEventRecord(ev.e0, st));
  bool fused = false;                                        // a9 at the end of the transport launch (when it can be)
  rc = launch_transport(ctx, seed, first, n, st, nullptr, n <= (1ull << 31) ? &fused : nullptr);
  if (rc != MCRT_OK) { ctx->spare.push_back(ev); return rc; }
  CU(cudaEventRecord(ev.e1, st));
  ctx->Ncum += n;
  ctx->Nglobal = ctx->Ncum;
  if (!fused) rc = launch_update(ctx, ctx->d_tally, ctx->Ncum, st);
  if (rc != MCRT_OK) { ctx->spare.push_back(ev); return rc; }
  CU(cudaEventRecord(ev.e2, st));
  ctx->pending.push_back(ev);
  ctx->last_stream = st;
  return MCRT_OK;
}

mcrt_status mcrt_transport_batch(mcrt_ctx* ctx, uint64_t seed, uint64_t first, uint64_t n, void* stream_) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->have_source) return fail(ctx, MCRT_ESTATE, "mcrt_transport_batch: grid, opacity and sources must be set first");
  cudaStream_t st = (cudaStream_t)stream_;
  BatchEvents ev;
  mcrt_status rc = begin_batch(ctx, &ev);
  if (rc != MCRT_OK) return rc;
  CU(cudaEventRecord(ev.e0, st));
  rc = launch_transport(ctx, seed, first, n, st);
  if (rc != MCRT_OK) { ctx->spare.push_back(ev); return rc; }
  CU(cudaEventRecord(ev.e1, st));
  CU(cudaEventRecord(ev.e2, st));
  ctx->pending.push_back(ev);
  ctx->Ncum += n;
  ctx->last_stream = st;
  return MCRT_OK;
}

mcrt_status mcrt_update_temperature(mcrt_ctx* ctx, const uint64_t* tally_sum, uint64_t n_cum, void* stream_) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->have_source) return fail(ctx, MCRT_ESTATE, "mcrt_update_temperature: grid, opacity and sources must be set first");
  cudaStream_t st = (cudaStream_t)stream_;
  ctx->Nglobal = tally_sum ? n_cum : ctx->Ncum;             // eps of mcrt_get_cell_energy = L_tot / packages of all ranks
  mcrt_status rc = launch_update(ctx, tally_sum ? (const unsigned long long*)tally_sum : ctx->d_tally,
                                 tally_sum ? n_cum : ctx->Ncum, st);
  ctx->last_stream = st;
  return rc;
}

int64_t mcrt_store_slots(const mcrt_ctx* ctx) { return ctx ? ctx->store_slots : -1; }
int64_t mcrt_delta_words(const mcrt_ctx* ctx) {
  if (!ctx) return -1;
  return ctx->store_slots * (ctx->pah ? 1 + (int64_t)ctx->nb : 1);
}

mcrt_status mcrt_transport_batch_delta(mcrt_ctx* ctx, uint64_t seed, uint64_t first, uint64_t n, uint32_t* delta_dev,
                                       void* stream_) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->have_source) return fail(ctx, MCRT_ESTATE, "mcrt_transport_batch_delta: grid, opacity and sources must be set first");
  if (!delta_dev) return fail(ctx, MCRT_EINVAL, "mcrt_transport_batch_delta: NULL delta buffer");
  cudaStream_t st = (cudaStream_t)stream_;
  BatchEvents ev;
  mcrt_status rc = begin_batch(ctx, &ev);
  if (rc != MCRT_OK) return rc;
  CU(cudaEventRecord(ev.e0, st));
  CU(cudaMemsetAsync(delta_dev, 0, sizeof(uint32_t) * (size_t)mcrt_delta_words(ctx), st));
  rc = launch_transport(ctx, seed, first, n, st, delta_dev);
  if (rc != MCRT_OK) { ctx->spare.push_back(ev); return rc; }
  CU(cudaEventRecord(ev.e1, st));
  CU(cudaEventRecord(ev.e2, st));
  ctx->pending.push_back(ev);
  ctx->Ncum += n;
  ctx->last_stream = st;
  return MCRT_OK;
}

mcrt_status mcrt_accumulate_update(mcrt_ctx* ctx, const uint32_t* delta_sum_dev, uint64_t n_cum, void* stream_) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->have_source) return fail(ctx, MCRT_ESTATE, "mcrt_accumulate_update: grid, opacity and sources must be set first");
  if (!delta_sum_dev || n_cum == 0) return fail(ctx, MCRT_EINVAL, "mcrt_accumulate_update: NULL delta / n_cum = 0");
  cudaStream_t st = (cudaStream_t)stream_;
  ctx->Nglobal = n_cum;
  if (ctx->pah) {                                            // the PAH's absorbed spectra of the batch, all ranks
    const long long nw = (long long)ctx->store_slots * ctx->nb;
    k_add_u32<<<(unsigned)std::min<long long>((nw + 1023) / 1024, (long long)ctx->sm_count * 16), 256, 0, st>>>(
        ctx->d_pah_cnt, delta_sum_dev + ctx->store_slots, nw);
    ctx->launches++;
    CU(cudaGetLastError());
  }
  mcrt_status rc = launch_update(ctx, ctx->d_tally, n_cum, st, delta_sum_dev);
  ctx->last_stream = st;
  return rc;
}

static mcrt_status sync_last(mcrt_ctx* ctx) {
  CU(cudaStreamSynchronize(ctx->last_stream));
  return MCRT_OK;
}

static mcrt_status copy_out(mcrt_ctx* ctx, void* dst, const void* src, size_t bytes, mcrt_mem mem) {
  CU(cudaMemcpyAsync(dst, src, bytes, mem == MCRT_DEVICE ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                     ctx->last_stream));
  CU(cudaStreamSynchronize(ctx->last_stream));
  return MCRT_OK;
}

mcrt_status mcrt_get_cell_energy(mcrt_ctx* ctx, uint64_t* n_abs_out, double* eps_out, mcrt_mem mem) {
  if (!ctx) return MCRT_EINVAL;
  if (!n_abs_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_cell_energy: NULL output");
  {
    const unsigned long long n_eps = ctx->Nglobal > ctx->Ncum ? ctx->Nglobal : ctx->Ncum;
    if (eps_out) *eps_out = n_eps ? ctx->Ltot / (double)n_eps : 0.0;
  }
  if (needs_reorder(ctx)) {                                  // storage order -> slot order (R22)
    unsigned long long* d_out = (unsigned long long*)n_abs_out;
    unsigned long long* tmp = nullptr;
    if (mem == MCRT_HOST) {
      if (!ctx->d_out_scratch) CU(mc_malloc(&ctx->d_out_scratch, 8 * (size_t)ctx->slots));
      tmp = (unsigned long long*)ctx->d_out_scratch; d_out = tmp;
    }
    mcrt_status rc = store_to_api_u64(ctx, ctx->d_tally, d_out, ctx->last_stream);
    if (rc != MCRT_OK) return rc;
    CU(cudaGetLastError());
    if (mem == MCRT_HOST) return copy_out(ctx, n_abs_out, tmp, 8 * (size_t)ctx->slots, MCRT_HOST);
    return sync_last(ctx);
  }
  return copy_out(ctx, n_abs_out, ctx->d_tally, 8 * (size_t)ctx->slots, mem);
}

mcrt_status mcrt_get_cell_temperature(mcrt_ctx* ctx, float* T_out, mcrt_mem mem) {
  if (!ctx) return MCRT_EINVAL;
  if (!T_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_cell_temperature: NULL output");
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_get_cell_temperature: opacity not set");
  float* d_T = T_out;
  float* tmp = nullptr;
  if (mem == MCRT_HOST) {
    if (!ctx->d_out_scratch) CU(mc_malloc(&ctx->d_out_scratch, 8 * (size_t)ctx->slots));
    tmp = (float*)ctx->d_out_scratch; d_T = tmp;
  }
  {
    mcrt_status rc = trow_to_api_T(ctx, d_T, ctx->last_stream);
    if (rc != MCRT_OK) return rc;
  }
  CU(cudaGetLastError());
  if (mem == MCRT_HOST) return copy_out(ctx, T_out, tmp, 4 * (size_t)ctx->slots, MCRT_HOST);
  return sync_last(ctx);
}

// Address of the current GPU's copy of g_noalloc_T (asked once per GPU; the caller holds g_noalloc_mutex).
static mcrt_status noalloc_T_array(mcrt_ctx* ctx, int dev, float** out) {
  if (!g_noalloc_T_ptr[dev]) {
    float* p = nullptr;
    CU(cudaGetSymbolAddress((void**)&p, g_noalloc_T));
    if (!p) return fail(ctx, MCRT_ECUDA, "mcrt_get_cell_temperature_noalloc: cudaGetSymbolAddress returned NULL");
    g_noalloc_T_ptr[dev] = p;
  }
  *out = g_noalloc_T_ptr[dev];
  return MCRT_OK;
}

// mcrt_get_cell_temperature for callers that cannot allocate device memory (include/mcrt.h says who): the same
// conversion kernels, writing into the library's own fixed array instead of a cudaMalloc'ed one.  No cudaMalloc /
// cudaFree / allocating CUDA call on this path; nothing in the array needs clearing (every float copied out is
// written first).  The lock is held until the copy to the host is complete, so calls never overlap on the GPU.
mcrt_status mcrt_get_cell_temperature_noalloc(mcrt_ctx* ctx, float* T_out_host) {
  if (!ctx) return MCRT_EINVAL;
  if (!T_out_host) return fail(ctx, MCRT_EINVAL, "mcrt_get_cell_temperature_noalloc: NULL output");
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_get_cell_temperature_noalloc: opacity not set");
  if (ctx->slots > kNoallocMaxSlots)
    return fail(ctx, MCRT_EINVAL, "mcrt_get_cell_temperature_noalloc: the grid has " + std::to_string(ctx->slots) +
                                      " leaf slots, the library's fixed array holds MCRT_NOALLOC_MAX_SLOTS = " +
                                      std::to_string(kNoallocMaxSlots) + " (use mcrt_get_cell_temperature, which allocates)");
  int dev = -1;
  CU(cudaGetDevice(&dev));
  if (dev != ctx->device)
    return fail(ctx, MCRT_ESTATE, "mcrt_get_cell_temperature_noalloc: the context lives on device " +
                                      std::to_string(ctx->device) + " but device " + std::to_string(dev) + " is current");
  if (dev < 0 || dev >= kNoallocMaxDevices)
    return fail(ctx, MCRT_EINVAL, "mcrt_get_cell_temperature_noalloc: device index beyond " + std::to_string(kNoallocMaxDevices - 1));
  std::lock_guard<std::mutex> lock(g_noalloc_mutex);
  float* d_T = nullptr;
  {
    mcrt_status rc = noalloc_T_array(ctx, dev, &d_T);
    if (rc != MCRT_OK) return rc;
  }
  {
    mcrt_status rc = trow_to_api_T(ctx, d_T, ctx->last_stream);
    if (rc != MCRT_OK) return rc;
  }
  CU(cudaGetLastError());
  return copy_out(ctx, T_out_host, d_T, 4 * (size_t)ctx->slots, MCRT_HOST);
}

mcrt_status mcrt_get_sed(mcrt_ctx* ctx, uint64_t* counts_out, mcrt_mem mem) {
  if (!ctx) return MCRT_EINVAL;
  if (!counts_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_sed: NULL output");
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_get_sed: opacity not set");
  return copy_out(ctx, counts_out, ctx->d_small + 1 + CNT_N, 8 * 3 * (size_t)ctx->nb, mem);
}

// ---- transiently heated PAH (row f2) --------------------------------------------------------------
static mcrt_status pah_reset_rows(mcrt_ctx* ctx) {
  const long long n = ctx->store_slots * (long long)ctx->nb;
  CU(cudaMemset(ctx->d_pah_cnt, 0, sizeof(uint32_t) * (size_t)n));
  k_pah_fill_rows<<<(unsigned)((n + 255) / 256), 256>>>(ctx->d_pah_cold, ctx->d_pah_cdf, ctx->store_slots, ctx->nb);
  ctx->launches++;
  CU(cudaGetLastError());
  return MCRT_OK;
}

mcrt_status mcrt_set_pah(mcrt_ctx* ctx, const mcrt_pah_desc* d) {
  if (!ctx) return MCRT_EINVAL;
  if (!d || !d->kabs_pah) return fail(ctx, MCRT_EINVAL, "mcrt_set_pah: NULL argument");
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_set_pah: call mcrt_set_opacity first");
  int K = d->n_Tp;
  double T_lo = d->T_lo, T_hi = d->T_hi, theta = d->theta_K;
  if (K == 0) { K = 128; T_lo = 5.0; T_hi = 1.0e4; }
  if (!(theta > 0)) theta = 500.0;
  if (d->n_C < 1 || !(d->mass_fraction > 0) || d->mass_fraction > 1 || K < 4 || K > 1024 || !(T_lo > 0) || !(T_hi > T_lo))
    return fail(ctx, MCRT_EINVAL, "mcrt_set_pah: n_C >= 1, 0 < mass_fraction <= 1, 4 <= n_Tp <= 1024, 0 < T_lo < T_hi");
  if ((double)ctx->store_slots * ctx->nb >= 4.0e9)
    return fail(ctx, MCRT_EINVAL, "mcrt_set_pah: leaf slots x n_bins must stay below 4e9 (per-leaf spectra)");
  CU(cudaDeviceSynchronize());
  free_pah(ctx);
  const int nb = ctx->nb;
  float* d_in = nullptr;
  struct Tmp { float*& a; ~Tmp() { mc_free(a); } } tmp{d_in};
  CU(mc_malloc(&d_in, 4 * (size_t)nb));
  CU(cudaMemcpy(d_in, d->kabs_pah, 4 * (size_t)nb, cudaMemcpyHostToDevice));
  CU(mc_malloc(&ctx->d_kabs_eq, 8 * (size_t)nb)); CU(mc_malloc(&ctx->d_pah_q, 4 * (size_t)nb));
  CU(mc_malloc(&ctx->d_pah_C, 8 * (size_t)nb)); CU(mc_malloc(&ctx->d_pah_E, 8 * (size_t)nb));
  CU(mc_malloc(&ctx->d_pah_T, 8 * (size_t)K)); CU(mc_malloc(&ctx->d_pah_U, 8 * (size_t)K));
  CU(mc_malloc(&ctx->d_pah_Lam, 8 * (size_t)K)); CU(mc_malloc(&ctx->d_pah_P, 8 * (size_t)K));
  CU(mc_malloc(&ctx->d_pah_W, 8 * (size_t)K * nb)); CU(mc_malloc(&ctx->d_pah_J, sizeof(int) * (size_t)K * K));
  CU(mc_malloc(&ctx->d_pah_W32, 4 * (size_t)K * nb));
  CU(mc_malloc(&ctx->d_pah_cold, 4 * (size_t)nb));
  CU(mc_malloc(&ctx->d_pah_cnt, sizeof(uint32_t) * (size_t)ctx->store_slots * nb));
  CU(mc_malloc(&ctx->d_pah_cdf, sizeof(float) * (size_t)ctx->store_slots * nb));
  k_pah_split<<<(nb + 127) / 128, 128>>>(nb, ctx->d_kabs, d_in, ctx->d_nu, d->n_C, d->mass_fraction, ctx->d_kabs_eq,
                                         ctx->d_pah_q, ctx->d_pah_C, ctx->d_pah_E);
  // the equilibrium tables from what is left for the grains in equilibrium (R35)
  k_build_emission_rows<<<ctx->nT, 128, 8 * (nb + 1)>>>(nb, ctx->nT, ctx->Tmin, ctx->Tmax, ctx->d_nu, ctx->d_dnu,
                                                        ctx->d_kabs_eq, ctx->d_lnQ, ctx->d_cdf);
  k_build_guide<<<kGuide / 256, 256>>>(ctx->d_lnQ, ctx->nT, ctx->d_guide);
  k_build_cdf_guide<<<ctx->nT, kCdfGuide>>>(ctx->d_cdf, nb, ctx->nT, ctx->d_cdf_guide);
  k_pah_states<<<K, 128>>>(nb, K, T_lo, T_hi, d->n_C, theta, ctx->d_nu, ctx->d_dnu, ctx->d_pah_C, ctx->d_pah_T,
                           ctx->d_pah_U, ctx->d_pah_Lam, ctx->d_pah_W, ctx->d_pah_W32);
  k_pah_thresholds<<<(K * K + 255) / 256, 256>>>(nb, K, ctx->d_pah_E, ctx->d_pah_U, ctx->d_pah_J);
  k_pah_cold_row<<<1, 32>>>(nb, ctx->d_pah_W, ctx->d_pah_cold);
  ctx->launches += 7;
  CU(cudaGetLastError());
  ctx->pahd.nC = d->n_C; ctx->pahd.K = K; ctx->pahd.nb = nb; ctx->pahd.fP = d->mass_fraction; ctx->pahd.theta = theta;
  ctx->pahd.E = ctx->d_pah_E; ctx->pahd.U = ctx->d_pah_U; ctx->pahd.Lam = ctx->d_pah_Lam; ctx->pahd.W = ctx->d_pah_W;
  ctx->pahd.J = ctx->d_pah_J; ctx->pahd.W32 = ctx->d_pah_W32;
  mcrt_status rc = pah_reset_rows(ctx);
  if (rc != MCRT_OK) return rc;
  CU(cudaDeviceSynchronize());
  ctx->pah = true;
  return MCRT_OK;
}

}  // extern "C" (templates follow)

// per-leaf rows of n_bins values: storage order -> the caller's slot order
template <typename T>
static mcrt_status rows_to_api(mcrt_ctx* ctx, const T* store, T* out, cudaStream_t st) {
  const int nb = ctx->nb;
  if (ctx->macro) {
    const long long nf3 = ctx->slots;
    k_rows_store_to_ext<T><<<(unsigned)((nf3 * nb + 255) / 256), 256, 0, st>>>(store + (size_t)ctx->store_n3 * nb, out, ctx->lay_fine, nf3, nb);
  } else {
    k_rows_store_to_ext<T><<<(unsigned)((ctx->n3 * nb + 255) / 256), 256, 0, st>>>(store, out, ctx->lay, ctx->n3, nb);
    if (ctx->slots > ctx->n3)
      CU(cudaMemcpyAsync(out + (size_t)ctx->n3 * nb, store + (size_t)ctx->store_n3 * nb,
                         sizeof(T) * (size_t)(ctx->slots - ctx->n3) * nb, cudaMemcpyDeviceToDevice, st));
  }
  ctx->launches++;
  CU(cudaGetLastError());
  return MCRT_OK;
}
template <typename T>
static mcrt_status get_rows(mcrt_ctx* ctx, const T* store, T* out, mcrt_mem mem) {
  const size_t bytes = sizeof(T) * (size_t)ctx->slots * ctx->nb;
  T* d_out = out;
  T* tmp = nullptr;
  struct Tmp { T*& a; ~Tmp() { mc_free(a); } } guard{tmp};
  if (mem == MCRT_HOST) { CU(mc_malloc(&tmp, bytes)); d_out = tmp; }
  mcrt_status rc = rows_to_api<T>(ctx, store, d_out, ctx->last_stream);
  if (rc != MCRT_OK) return rc;
  if (mem == MCRT_HOST) return copy_out(ctx, out, tmp, bytes, MCRT_HOST);
  return sync_last(ctx);
}

extern "C" {

mcrt_status mcrt_get_pah_absorbed(mcrt_ctx* ctx, uint32_t* counts_out, mcrt_mem mem) {
  if (!ctx) return MCRT_EINVAL;
  if (!counts_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_pah_absorbed: NULL output");
  if (!ctx->pah) return fail(ctx, MCRT_ESTATE, "mcrt_get_pah_absorbed: no PAH declared (mcrt_set_pah)");
  return get_rows<uint32_t>(ctx, ctx->d_pah_cnt, counts_out, mem);
}

mcrt_status mcrt_get_pah_emission_cdf(mcrt_ctx* ctx, float* cdf_out, mcrt_mem mem) {
  if (!ctx) return MCRT_EINVAL;
  if (!cdf_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_pah_emission_cdf: NULL output");
  if (!ctx->pah) return fail(ctx, MCRT_ESTATE, "mcrt_get_pah_emission_cdf: no PAH declared (mcrt_set_pah)");
  return get_rows<float>(ctx, ctx->d_pah_cdf, cdf_out, mem);
}

// storage slot of a leaf slot of the caller's order (R22)
static long long storage_slot_of(const mcrt_ctx* ctx, long long api) {
  if (ctx->macro) {
    const int N = ctx->n_fine;
    return ctx->store_n3 + slot_of(ctx->lay_fine, (int)(api % N), (int)((api / N) % N), (int)(api / ((long long)N * N)));
  }
  if (api >= ctx->n3) return ctx->store_n3 + (api - ctx->n3);
  const int N = ctx->N;
  return slot_of(ctx->lay, (int)(api % N), (int)((api / N) % N), (int)(api / ((long long)N * N)));
}

mcrt_status mcrt_get_pah_temperature_distribution(mcrt_ctx* ctx, int64_t leaf_slot, double* T_out, double* P_out) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->pah) return fail(ctx, MCRT_ESTATE, "mcrt_get_pah_temperature_distribution: no PAH declared (mcrt_set_pah)");
  if (leaf_slot < 0 || leaf_slot >= ctx->slots || !P_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_pah_temperature_distribution: bad slot / NULL");
  const int K = ctx->pahd.K;
  const unsigned long long n_cum = ctx->Nglobal > ctx->Ncum ? ctx->Nglobal : ctx->Ncum;
  std::vector<double> P(K, 0.0);
  P[0] = 1.0;                                                // nothing absorbed yet: the ground state
  CU(cudaMemcpyAsync(ctx->d_pah_P, P.data(), 8 * (size_t)K, cudaMemcpyHostToDevice, ctx->last_stream));
  if (n_cum) {
    mcrt_status rc = launch_pah_update(ctx, n_cum, ctx->last_stream, storage_slot_of(ctx, leaf_slot));
    if (rc != MCRT_OK) return rc;
  }
  mcrt_status rc = copy_out(ctx, P_out, ctx->d_pah_P, 8 * (size_t)K, MCRT_HOST);
  if (rc != MCRT_OK) return rc;
  if (T_out) return copy_out(ctx, T_out, ctx->d_pah_T, 8 * (size_t)K, MCRT_HOST);
  return MCRT_OK;
}

// ---- combined / asynchronous read-out ----------------------------------------------------------
mcrt_status mcrt_results_begin(mcrt_ctx* ctx, const mcrt_results* out, mcrt_mem mem, int32_t* ticket) {
  if (!ctx) return MCRT_EINVAL;
  if (!out || !ticket) return fail(ctx, MCRT_EINVAL, "mcrt_results_begin: NULL argument");
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_results_begin: opacity not set");
  const int s = ctx->next_ticket;
  mcrt_ctx::Ticket& t = ctx->tickets[s];
  if (t.busy) return fail(ctx, MCRT_ESTATE, "mcrt_results_begin: both tickets are in flight (call mcrt_results_wait)");
  cudaStream_t st = ctx->last_stream;
  if (!ctx->copy_stream) CU(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking));
  if (!t.ev_snap) { CU(cudaEventCreateWithFlags(&t.ev_snap, cudaEventDisableTiming)); CU(cudaEventCreateWithFlags(&t.ev_done, cudaEventDisableTiming)); }
  const size_t n_small = 1 + CNT_N + 4 * (size_t)ctx->nb;
  const bool host = mem == MCRT_HOST;
  // 1. snapshot on the batches' stream (the next batch may start right behind it)
  unsigned long long* abs_dst = nullptr;
  float* T_dst = nullptr;
  if (out->n_abs) {
    if (host && !t.snap_abs) CU(mc_malloc(&t.snap_abs, 8 * (size_t)ctx->slots));
    abs_dst = host ? t.snap_abs : (unsigned long long*)out->n_abs;
    if (needs_reorder(ctx)) {
      mcrt_status rc = store_to_api_u64(ctx, ctx->d_tally, abs_dst, st);
      if (rc != MCRT_OK) return rc;
    } else {
      CU(cudaMemcpyAsync(abs_dst, ctx->d_tally, 8 * (size_t)ctx->slots, cudaMemcpyDeviceToDevice, st));
    }
  }
  if (out->T) {
    if (host && !t.snap_T) CU(mc_malloc(&t.snap_T, 4 * (size_t)ctx->slots));
    T_dst = host ? t.snap_T : out->T;
    mcrt_status rc = trow_to_api_T(ctx, T_dst, st);
    if (rc != MCRT_OK) return rc;
  }
  if (!t.snap_small) { CU(mc_malloc(&t.snap_small, 8 * n_small)); }
  CU(cudaMemcpyAsync(t.snap_small, ctx->d_small, 8 * n_small, cudaMemcpyDeviceToDevice, st));
  CU(cudaGetLastError());
  CU(cudaEventRecord(t.ev_snap, st));
  // 2. copies out on the context's own stream
  cudaStream_t cs = ctx->copy_stream;
  CU(cudaStreamWaitEvent(cs, t.ev_snap, 0));
  if (host) {
    if (out->n_abs) CU(cudaMemcpyAsync(out->n_abs, t.snap_abs, 8 * (size_t)ctx->slots, cudaMemcpyDeviceToHost, cs));
    if (out->T) CU(cudaMemcpyAsync(out->T, t.snap_T, 4 * (size_t)ctx->slots, cudaMemcpyDeviceToHost, cs));
  }
  if (!t.h_small) CU(cudaMallocHost(&t.h_small, 8 * 8192 * 5));     // n_bins <= 4096
  CU(cudaMemcpyAsync(t.h_small, t.snap_small, 8 * n_small, cudaMemcpyDeviceToHost, cs));
  if (!host) {
    if (out->sed) CU(cudaMemcpyAsync(out->sed, t.snap_small + 1 + CNT_N, 8 * 3 * (size_t)ctx->nb, cudaMemcpyDeviceToDevice, cs));
    if (out->emitted_per_bin)
      CU(cudaMemcpyAsync(out->emitted_per_bin, t.snap_small + 1 + CNT_N + 3 * (size_t)ctx->nb, 8 * (size_t)ctx->nb, cudaMemcpyDeviceToDevice, cs));
  }
  CU(cudaEventRecord(t.ev_done, cs));
  if (out->eps) {
    const unsigned long long n_eps = ctx->Nglobal > ctx->Ncum ? ctx->Nglobal : ctx->Ncum;
    *out->eps = n_eps ? ctx->Ltot / (double)n_eps : 0.0;
  }
  t.counters = out->counters; t.mem = mem;
  t.sed = host ? out->sed : nullptr; t.emitted = host ? out->emitted_per_bin : nullptr;
  t.busy = true;
  *ticket = s;
  ctx->next_ticket = s ^ 1;
  return MCRT_OK;
}

mcrt_status mcrt_results_wait(mcrt_ctx* ctx, int32_t ticket) {
  if (!ctx) return MCRT_EINVAL;
  if (ticket < 0 || ticket > 1 || !ctx->tickets[ticket].busy) return fail(ctx, MCRT_EINVAL, "mcrt_results_wait: no such ticket in flight");
  mcrt_ctx::Ticket& t = ctx->tickets[ticket];
  CU(cudaEventSynchronize(t.ev_done));
  const unsigned long long* h = t.h_small + 1;
  if (t.counters) {
    t.counters->emitted = h[CNT_EMITTED]; t.counters->escaped = h[CNT_ESCAPED]; t.counters->lost = h[CNT_LOST];
    t.counters->absorptions = h[CNT_ABS]; t.counters->scatterings = h[CNT_SCA]; t.counters->flights = h[CNT_FLIGHTS];
    t.counters->crossings = h[CNT_CROSS];
  }
  if (t.sed) std::memcpy(t.sed, h + CNT_N, 8 * 3 * (size_t)ctx->nb);
  if (t.emitted) std::memcpy(t.emitted, h + CNT_N + 3 * (size_t)ctx->nb, 8 * (size_t)ctx->nb);
  t.busy = false;
  return MCRT_OK;
}

mcrt_status mcrt_get_results(mcrt_ctx* ctx, const mcrt_results* out, mcrt_mem mem) {
  int32_t ticket = -1;
  mcrt_status rc = mcrt_results_begin(ctx, out, mem, &ticket);
  if (rc != MCRT_OK) return rc;
  return mcrt_results_wait(ctx, ticket);
}

mcrt_status mcrt_set_observer(mcrt_ctx* ctx, const mcrt_observer_desc* d) {
  if (!ctx) return MCRT_EINVAL;
  if (!d) return fail(ctx, MCRT_EINVAL, "mcrt_set_observer: NULL argument");
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_set_observer: call mcrt_set_opacity first");
  if (d->n_mu < 0 || d->n_mu > 4096 || d->n_pix < 0 || d->n_pix > 8192)
    return fail(ctx, MCRT_EINVAL, "mcrt_set_observer: n_mu must be 0..4096, n_pix 0..8192");
  double o[3] = {0, 0, 1}, e1[3] = {1, 0, 0}, e2[3] = {0, 1, 0};
  if (d->n_pix > 0) {
    const double n = std::sqrt(d->dir[0] * d->dir[0] + d->dir[1] * d->dir[1] + d->dir[2] * d->dir[2]);
    if (!(n > 0) || !(d->half_width > 0) || !(d->half_angle_deg > 0) || d->half_angle_deg > 180)
      return fail(ctx, MCRT_EINVAL, "mcrt_set_observer: dir must be non-zero, half_width > 0, 0 < half_angle_deg <= 180");
    for (int a = 0; a < 3; ++a) o[a] = d->dir[a] / n;
    // e1 = z x o normalised (R34); within 2.6 degrees of the pole, where that is ill-conditioned, e1 = the
    // component of x normal to o, normalised (Gram-Schmidt; exactly x for o along z)
    if (std::fabs(o[2]) < 0.999) {
      const double q = std::sqrt(o[0] * o[0] + o[1] * o[1]);
      e1[0] = -o[1] / q; e1[1] = o[0] / q; e1[2] = 0;
    } else {
      const double v[3] = {1.0 - o[0] * o[0], -o[0] * o[1], -o[0] * o[2]};
      const double q = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
      for (int a = 0; a < 3; ++a) e1[a] = v[a] / q;
    }
    e2[0] = o[1] * e1[2] - o[2] * e1[1];                    // e2 = o x e1
    e2[1] = o[2] * e1[0] - o[0] * e1[2];
    e2[2] = o[0] * e1[1] - o[1] * e1[0];
  }
  CU(cudaDeviceSynchronize());
  free_observer(ctx);
  if (d->n_mu > 0) {
    CU(mc_malloc(&ctx->obs.sed_mu, 8 * (size_t)d->n_mu * 3 * ctx->nb));
    CU(cudaMemset(ctx->obs.sed_mu, 0, 8 * (size_t)d->n_mu * 3 * ctx->nb));
  }
  if (d->n_pix > 0) {
    CU(mc_malloc(&ctx->obs.image, 8 * (size_t)d->n_pix * d->n_pix));
    CU(cudaMemset(ctx->obs.image, 0, 8 * (size_t)d->n_pix * d->n_pix));
  }
  ctx->obs.n_mu = d->n_mu; ctx->obs.n_pix = d->n_pix;
  ctx->obs.bin_lo = d->bin_lo; ctx->obs.bin_hi = d->bin_hi < 0 ? ctx->nb - 1 : d->bin_hi;
  for (int a = 0; a < 3; ++a) { ctx->obs.o[a] = (float)o[a]; ctx->obs.e1[a] = (float)e1[a]; ctx->obs.e2[a] = (float)e2[a]; }
  ctx->obs.cos_alpha = d->n_pix > 0 ? (float)std::cos(d->half_angle_deg * 3.14159265358979323846 / 180.0) : 1.f;
  ctx->obs.half_width = d->n_pix > 0 ? (float)(d->half_width / ctx->root_size) : 1.f;
  return MCRT_OK;
}

mcrt_status mcrt_get_sed_mu(mcrt_ctx* ctx, uint64_t* counts_out, mcrt_mem mem) {
  if (!ctx) return MCRT_EINVAL;
  if (!counts_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_sed_mu: NULL output");
  if (!ctx->obs.sed_mu) return fail(ctx, MCRT_ESTATE, "mcrt_get_sed_mu: no inclination bins set (mcrt_set_observer)");
  return copy_out(ctx, counts_out, ctx->obs.sed_mu, 8 * (size_t)ctx->obs.n_mu * 3 * ctx->nb, mem);
}

mcrt_status mcrt_get_image(mcrt_ctx* ctx, uint64_t* counts_out, mcrt_mem mem) {
  if (!ctx) return MCRT_EINVAL;
  if (!counts_out) return fail(ctx, MCRT_EINVAL, "mcrt_get_image: NULL output");
  if (!ctx->obs.image) return fail(ctx, MCRT_ESTATE, "mcrt_get_image: no image set (mcrt_set_observer)");
  return copy_out(ctx, counts_out, ctx->obs.image, 8 * (size_t)ctx->obs.n_pix * ctx->obs.n_pix, mem);
}

mcrt_status mcrt_get_counters(mcrt_ctx* ctx, mcrt_counters* out, uint64_t* emitted_per_bin) {
  if (!ctx) return MCRT_EINVAL;
  if (!out) return fail(ctx, MCRT_EINVAL, "mcrt_get_counters: NULL output");
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_get_counters: opacity not set");
  unsigned long long h[CNT_N];
  mcrt_status rc = copy_out(ctx, h, ctx->d_small + 1, 8 * CNT_N, MCRT_HOST);
  if (rc != MCRT_OK) return rc;
  out->emitted = h[CNT_EMITTED]; out->escaped = h[CNT_ESCAPED]; out->lost = h[CNT_LOST];
  out->absorptions = h[CNT_ABS]; out->scatterings = h[CNT_SCA]; out->flights = h[CNT_FLIGHTS];
  out->crossings = h[CNT_CROSS];
  if (emitted_per_bin)
    return copy_out(ctx, emitted_per_bin, ctx->d_small + 1 + CNT_N + 3 * (size_t)ctx->nb, 8 * (size_t)ctx->nb, MCRT_HOST);
  return MCRT_OK;
}

mcrt_status mcrt_reset_tallies(mcrt_ctx* ctx, int32_t what) {
  if (!ctx) return MCRT_EINVAL;
  CU(cudaStreamSynchronize(ctx->last_stream));
  if ((what & 1) && ctx->d_small) CU(cudaMemset(ctx->d_small, 0, 8 * (1 + CNT_N + 4 * (size_t)ctx->nb)));
  if ((what & 1) && ctx->obs.sed_mu) CU(cudaMemset(ctx->obs.sed_mu, 0, 8 * (size_t)ctx->obs.n_mu * 3 * ctx->nb));
  if ((what & 1) && ctx->obs.image) CU(cudaMemset(ctx->obs.image, 0, 8 * (size_t)ctx->obs.n_pix * ctx->obs.n_pix));
  if (what & 2) {
    CU(cudaMemset(ctx->d_tally, 0, 8 * (size_t)ctx->store_slots));
    CU(cudaMemset(ctx->d_trow, 0, 4 * (size_t)ctx->store_slots));
    ctx->Ncum = 0;
    ctx->Nglobal = 0;
    if (ctx->pah) { mcrt_status rc = pah_reset_rows(ctx); if (rc != MCRT_OK) return rc; CU(cudaDeviceSynchronize()); }
  }
  return MCRT_OK;
}

mcrt_status mcrt_set_launch(mcrt_ctx* ctx, int32_t threads, int32_t blocks_per_sm) {
  if (!ctx) return MCRT_EINVAL;
  if (threads < 0 || threads > 256 || (threads % 32) != 0 || blocks_per_sm < 0 || blocks_per_sm > 32)
    return fail(ctx, MCRT_EINVAL, "mcrt_set_launch: threads must be a multiple of 32 up to 256, blocks_per_sm <= 32");
  if (threads) ctx->threads = threads;
  ctx->blocks_per_sm = blocks_per_sm;                        // 0 = automatic
  return MCRT_OK;
}

mcrt_status mcrt_set_walk_quorum(mcrt_ctx* ctx, int32_t quorum) {
  if (!ctx) return MCRT_EINVAL;
  if (quorum < 0 || quorum > 32) return fail(ctx, MCRT_EINVAL, "mcrt_set_walk_quorum: quorum must be 0..32");
  ctx->quorum = quorum;
  return MCRT_OK;
}

mcrt_status mcrt_set_tail_mode(mcrt_ctx* ctx, int32_t mode) {
  if (!ctx) return MCRT_EINVAL;
  if (mode < -1 || mode > 3) return fail(ctx, MCRT_EINVAL, "mcrt_set_tail_mode: -1 (automatic) or a combination of bits 0 and 1");
  ctx->tail_mode = mode;
  return MCRT_OK;
}

mcrt_status mcrt_set_region_sweeps(mcrt_ctx* ctx, int32_t sweeps, int32_t rx, int32_t ry, int32_t rz) {
  if (!ctx) return MCRT_EINVAL;
  if (sweeps < -1 || sweeps > 30) return fail(ctx, MCRT_EINVAL, "mcrt_set_region_sweeps: -1 (automatic), 0 (off) or 1..30");
  if (rx | ry | rz) {                                        // a new region shape: the marked tables are rebuilt
    const int shape[3] = {rx, ry, rz};
    if (!ctx->region_cells[0]) return fail(ctx, MCRT_ESTATE, "mcrt_set_region_sweeps: this grid is not swept (single-level, brick layout, >= 256^3)");
    long long nreg = 1;
    for (int a = 0; a < 3; ++a) {
      if (shape[a] < 8 || shape[a] % 8 || ctx->N % shape[a]) return fail(ctx, MCRT_EINVAL, "mcrt_set_region_sweeps: region edges must be multiples of 8 that divide n_root");
      nreg *= ctx->N / shape[a];
    }
    if (nreg < 2 || nreg > 4096) return fail(ctx, MCRT_EINVAL, "mcrt_set_region_sweeps: 2..4096 regions");
    CU(cudaDeviceSynchronize());
    std::vector<int> lut(6 * (size_t)ctx->N);
    CU(cudaMemcpy(lut.data(), ctx->d_lut, sizeof(int) * lut.size(), cudaMemcpyDeviceToHost));
    mcrt_status rc = build_region_tables(ctx, lut.data(), shape);
    if (rc != MCRT_OK) return rc;
  }
  ctx->region_sweeps = sweeps;
  return MCRT_OK;
}

mcrt_status mcrt_get_region_sweep_counts(mcrt_ctx* ctx, uint32_t* suspended_out, int32_t cap, int32_t* n_out) {
  if (!ctx) return MCRT_EINVAL;
  if (!suspended_out || !n_out || cap < 0) return fail(ctx, MCRT_EINVAL, "mcrt_get_region_sweep_counts: bad arguments");
  *n_out = 0;
  if (!ctx->d_swcnt) return MCRT_OK;                         // no batch was swept yet
  const int n = cap < 32 ? cap : 32;
  mcrt_status rc = copy_out(ctx, suspended_out, ctx->d_swcnt, sizeof(uint32_t) * (size_t)n, MCRT_HOST);
  if (rc != MCRT_OK) return rc;
  *n_out = n;
  return MCRT_OK;
}

mcrt_status mcrt_set_density_staging(mcrt_ctx* ctx, int32_t mode) {
  if (!ctx) return MCRT_EINVAL;
  if (mode < 0 || mode > 2) return fail(ctx, MCRT_EINVAL, "mcrt_set_density_staging: mode must be 0 (automatic), 1 (off) or 2 (also one bit per cell)");
  ctx->dens_off = mode;
  if (mode == 2) return prepare_density_bits(ctx);
  return MCRT_OK;
}

int32_t mcrt_density_staging(const mcrt_ctx* ctx) { return ctx ? staging_mode(ctx) : -1; }

mcrt_status mcrt_set_cdf_guide(mcrt_ctx* ctx, int32_t on) {
  if (!ctx) return MCRT_EINVAL;
  ctx->cdf_guide_off = on ? 0 : 1;
  return MCRT_OK;
}

mcrt_status mcrt_set_source_order(mcrt_ctx* ctx, int32_t mode) {
  if (!ctx) return MCRT_EINVAL;
  if (mode < -1 || mode > 2) return fail(ctx, MCRT_EINVAL, "mcrt_set_source_order: mode must be -1, 0, 1 or 2");
  ctx->order_by_source = mode;
  return MCRT_OK;
}

mcrt_status mcrt_get_batch_times(mcrt_ctx* ctx, float* transport_ms, float* update_ms, int32_t cap, int32_t* n_out) {
  if (!ctx) return MCRT_EINVAL;
  if (!n_out || cap < 0) return fail(ctx, MCRT_EINVAL, "mcrt_get_batch_times: bad arguments");
  int n = 0;
  for (auto& b : ctx->pending) {
    CU(cudaEventSynchronize(b.e2));
    if (n < cap) {
      float a = 0, c = 0;
      CU(cudaEventElapsedTime(&a, b.e0, b.e1));
      CU(cudaEventElapsedTime(&c, b.e1, b.e2));
      if (transport_ms) transport_ms[n] = a;
      if (update_ms) update_ms[n] = c;
      ++n;
    }
    ctx->spare.push_back(b);
  }
  ctx->pending.clear();
  *n_out = n;
  return MCRT_OK;
}

mcrt_status mcrt_get_tables(mcrt_ctx* ctx, float* opac, float* lnQ, float* cdf) {
  if (!ctx) return MCRT_EINVAL;
  if (!ctx->have_opacity) return fail(ctx, MCRT_ESTATE, "mcrt_get_tables: opacity not set");
  if (opac) CU(cudaMemcpy(opac, ctx->d_opac, 16 * (size_t)ctx->nb, cudaMemcpyDeviceToHost));
  if (lnQ) CU(cudaMemcpy(lnQ, ctx->d_lnQ, 4 * (size_t)ctx->nT, cudaMemcpyDeviceToHost));
  if (cdf) CU(cudaMemcpy(cdf, ctx->d_cdf, 4 * (size_t)ctx->nT * ctx->nb, cudaMemcpyDeviceToHost));
  return MCRT_OK;
}

int64_t mcrt_kernel_launches(const mcrt_ctx* ctx) { return ctx ? ctx->launches : -1; }

int64_t mcrt_debug_violations(void) {
#ifdef MCRT_CHECKS
  unsigned long long v = 0;
  if (cudaDeviceSynchronize() != cudaSuccess) return -2;
  if (cudaMemcpyFromSymbol(&v, g_mcrt_violations, sizeof(v)) != cudaSuccess) return -2;
  return (int64_t)v;
#else
  return -1;
#endif
}

__global__ void k_philox_blocks(uint32_t k0, uint32_t k1, const uint32_t* __restrict__ ctr,
                                uint32_t* __restrict__ out, long long n) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  uint32_t x[4];
  philox4x32_10(k0, k1, ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], x);
  out[4 * i] = x[0]; out[4 * i + 1] = x[1]; out[4 * i + 2] = x[2]; out[4 * i + 3] = x[3];
}

mcrt_status mcrt_philox_blocks(const uint32_t* key2, const uint32_t* ctr, uint32_t* out, int64_t n) {
  mcrt_ctx* ctx = nullptr;
  if (!key2 || !ctr || !out || n < 0) return fail(nullptr, MCRT_EINVAL, "mcrt_philox_blocks: bad arguments");
  if (n == 0) return MCRT_OK;
  uint32_t *d_c = nullptr, *d_o = nullptr;
  struct Tmp { uint32_t*& a; uint32_t*& b; ~Tmp() { mc_free(a); mc_free(b); } } tmp{d_c, d_o};
  CU(mc_malloc(&d_c, 16 * (size_t)n)); CU(mc_malloc(&d_o, 16 * (size_t)n));
  CU(cudaMemcpy(d_c, ctr, 16 * (size_t)n, cudaMemcpyHostToDevice));
  k_philox_blocks<<<(unsigned)((n + 255) / 256), 256>>>(key2[0], key2[1], d_c, d_o, n);
  CU(cudaGetLastError());
  CU(cudaMemcpy(out, d_o, 16 * (size_t)n, cudaMemcpyDeviceToHost));
  return MCRT_OK;
}

__global__ void k_uniforms(const uint32_t* __restrict__ w, float* __restrict__ u, double* __restrict__ ud,
                           float* __restrict__ tau, long long n) {
  long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  u[i] = u01(w[i]); ud[i] = u01d(w[i]); tau[i] = -logf(u01(w[i]));
}

mcrt_status mcrt_uniforms(const uint32_t* words, float* u, double* ud, float* tau, int64_t n) {
  mcrt_ctx* ctx = nullptr;
  if (!words || !u || !ud || !tau || n < 0) return fail(nullptr, MCRT_EINVAL, "mcrt_uniforms: bad arguments");
  if (n == 0) return MCRT_OK;
  uint32_t* d_w = nullptr; float *d_u = nullptr, *d_t = nullptr; double* d_ud = nullptr;
  struct Tmp { uint32_t*& a; float*& b; float*& c; double*& d; ~Tmp() { mc_free(a); mc_free(b); mc_free(c); mc_free(d); } } tmp{d_w, d_u, d_t, d_ud};
  CU(mc_malloc(&d_w, 4 * (size_t)n)); CU(mc_malloc(&d_u, 4 * (size_t)n)); CU(mc_malloc(&d_t, 4 * (size_t)n));
  CU(mc_malloc(&d_ud, 8 * (size_t)n));
  CU(cudaMemcpy(d_w, words, 4 * (size_t)n, cudaMemcpyHostToDevice));
  k_uniforms<<<(unsigned)((n + 255) / 256), 256>>>(d_w, d_u, d_ud, d_t, n);
  CU(cudaGetLastError());
  CU(cudaMemcpy(u, d_u, 4 * (size_t)n, cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(ud, d_ud, 8 * (size_t)n, cudaMemcpyDeviceToHost));
  CU(cudaMemcpy(tau, d_t, 4 * (size_t)n, cudaMemcpyDeviceToHost));
  return MCRT_OK;
}

mcrt_status mcrt_gather_calibrate(uint64_t footprint_bytes, uint64_t n_gathers, double* gathers_per_s,
                                  double* seconds, void* stream_) {
  mcrt_ctx* ctx = nullptr;
  if (!gathers_per_s || footprint_bytes < 4 || footprint_bytes > (16ull << 30) || n_gathers == 0)
    return fail(nullptr, MCRT_EINVAL, "mcrt_gather_calibrate: bad arguments (footprint 4 B .. 16 GiB, n_gathers > 0)");
  int dev = 0, sms = 0;
  CU(cudaGetDevice(&dev));
  CU(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  cudaStream_t st = (cudaStream_t)stream_;
  const uint32_t n_elems = (uint32_t)(footprint_bytes / 4);
  float *d_a = nullptr, *d_sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  struct Tmp { float*& a; float*& b; cudaEvent_t& e0; cudaEvent_t& e1;
               ~Tmp() { mc_free(a); mc_free(b); if (e0) cudaEventDestroy(e0); if (e1) cudaEventDestroy(e1); } } tmp{d_a, d_sink, e0, e1};
  CU(mc_malloc(&d_a, 4 * (size_t)n_elems));
  CU(mc_malloc(&d_sink, 4));
  CU(cudaMemsetAsync(d_a, 0, 4 * (size_t)n_elems, st));
  CU(cudaEventCreate(&e0)); CU(cudaEventCreate(&e1));
  const unsigned blocks = (unsigned)sms * 8u, threads = 256u;
  const uint64_t per_turn = 4ull * blocks * threads;
  uint32_t turns = (uint32_t)((n_gathers + per_turn - 1) / per_turn);
  if (turns < 1) turns = 1;
  k_gather_calibrate<<<blocks, threads, 0, st>>>(d_a, n_elems, turns < 16 ? turns : 16, d_sink);   // warm-up
  CU(cudaEventRecord(e0, st));
  k_gather_calibrate<<<blocks, threads, 0, st>>>(d_a, n_elems, turns, d_sink);
  CU(cudaEventRecord(e1, st));
  CU(cudaGetLastError());
  CU(cudaEventSynchronize(e1));
  float ms = 0.f;
  CU(cudaEventElapsedTime(&ms, e0, e1));
  const double sec = (double)ms * 1e-3;
  *gathers_per_s = sec > 0 ? (double)turns * (double)per_turn / sec : 0.0;
  if (seconds) *seconds = sec;
  return MCRT_OK;
}

int64_t mcrt_release_cached_memory(void) {
  McState& S = mc_state();
  std::lock_guard<std::mutex> lock(S.mutex);
  return (int64_t)mc_release_cache_locked(S);
}

const char* mcrt_last_error(const mcrt_ctx* ctx) { return ctx ? ctx->err.c_str() : g_err.c_str(); }

}  // extern "C"
