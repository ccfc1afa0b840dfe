// transport_u.cuh -- the sm_100a transport kernel: rows a1..a8 of SURVEY.md 8(a).
// One photon package per thread, persistent threads with lane refill, for single-level grids
// (template TL = false) and for two-level grids of cubes and subcubes (TL = true, PAPER.md L23
// "the cubes are further divided into subcubes (cells)").  DESIGN.md section 6.
//
//  * A package lives in registers and is never located from a floating-point position.  The cell
//    walk keeps ABSOLUTE path lengths along the current flight: t_a = path length at which the
//    package meets the next face of its leaf on axis a, tcur = path length so far.  One crossing
//    is tnext = min(t_x,t_y,t_z); dtau = rho*kappa*(tnext - tcur); the axis whose t equals tnext
//    (ties -> lowest axis, R21) advances by its pitch 1/|d_a| (times 1/S inside a refined cube).
//  * The leaf's storage slot is advanced by a per-axis DELTA table held in shared memory
//    (slot(ix,iy,iz) = A_x(ix) + A_y(iy) + A_z(iz) is separable, so the delta of a step depends
//    on one coordinate only).  The tables make the memory layout of the root grid a host decision
//    -- x-fastest, or 8^3 bricks in Morton order -- and mark the step that leaves the grid
//    (kLutEscape), so the hot loop has no bounds check and no index arithmetic beyond one add.
//    Per axis there is a forward and a reversed table, so a table cursor always moves by +1
//    whatever the direction's sign.
//  * Two-level grids use the SAME step: inside a refined cube the three cursors point into a tiny
//    second table (per axis and direction S entries +-S^a, the last one = kLutLeave) and the pitch
//    is 1/(S|d_a|); the root cursors, the root slot and the refined-cube number wait in five more
//    registers.  A step that reads kLutLeave takes the root table's delta, requests the new root
//    cube's entry and keeps walking at the sub level (the subcube index on the exit axis wraps,
//    the other two carry over: the faces of neighbouring refined cubes line up).  The density array
//    doubles as the two-level index: if the entry that comes back has its
//    sign bit set it names a refined cube (by its first leaf slot) and the leaf slot just moves to that cube
//    (integer arithmetic only); if not, the package has left the refined region and its exits move
//    out to the faces of the root cube.  A package that meets a marker at the root level descends
//    into the subcube its remaining distances to the root faces select.  Root-level and sub-level
//    lanes of a warp therefore run one instruction stream; the transitions between refined cubes
//    cost a handful of predicated instructions, only entering / leaving the refined REGION diverges.
//  * The density of the NEXT leaf is requested before the optical-depth test of the current one
//    (the geometric walk does not depend on rho), taking the gather latency off the dependent chain.
//  * Small problems keep their density ON CHIP (template DENS): a single-level grid of up to 40 KB
//    is copied into every block's shared memory as it is (DENS = 1: C0's 16^3), a grid with only
//    two distinct densities as ONE BIT per cell (DENS = 2: the uniform spheres, 64^3 = 32 KB), by
//    one cp.async.bulk (TMA) per block.  A crossing then costs a shared-memory read instead of an
//    L1TEX wavefront and an L2 round trip: this lifts the scattered-gather ceiling and shortens the
//    end-of-batch tail, where a lone package's crossing latency is all there is.
//  * MACRO: a single-level grid whose density is piecewise uniform (a sphere in vacuum) is run as a
//    two-level one: N/M macro cubes per axis, the M^3 cells of each behind the macro array.  A macro
//    cube whose cells all hold the same density is crossed in ONE step (the sum of equal per-cell
//    optical depths is the optical depth of the whole chord; empty space is skipped the same way);
//    a mixed cube carries the marker and is walked cell by cell.  Tallies and temperatures stay per
//    cell: an absorption inside a uniform cube is booked on the cell the interaction point lies in.
//    Cell crossings are not counted step by step there but from the cell coordinates at the two
//    ends of every flight (motion is monotonic per axis, so a flight crosses |F_end - F_start|
//    cell faces on each axis): "a kernel that skips empty space must add the skipped leaf count
//    arithmetically".
//  * REGION: grids far larger than the L2 (C4's 512^3) are swept region by region.  The root delta tables
//    carry a marker (kLutRegion) on every step that crosses a region boundary (regions of 128 x 128 x 128 cells
//    by default);
//    a package that takes such a step is SUSPENDED: its state (48 bytes) goes to a record indexed by its
//    package number and the number is appended, with the region it entered, to the list of the next sweep.
//    Between sweeps the list is grouped by region, so the packages in flight at any time sit in one or two
//    regions whose density the L2 holds: the walk's gathers become L2 hits instead of DRAM bursts.  After a
//    few sweeps the stragglers are finished by one sweep without markers.  Integer tallies and exact
//    restoration of the state make the result identical to the unswept run.
//  * The walk loop runs until fewer than `quorum` lanes of the warp are still walking; then all
//    stopped lanes go through ONE event pass (escape tally -> refill from the work queue ->
//    emission / scattering / absorption+re-emission -> new flight).  Emission and re-emission
//    share one instruction stream (Philox block -> CDF search -> isotropic direction).
#pragma once
#include <climits>
#include <cooperative_groups.h>
#include "tables.cuh"
#include "transport.cuh"

namespace mcrt {

// ---- storage layouts of a cubic array of N^3 cells (host and device) ----------------------------
struct LayoutU {
  int N;          // cells per axis
  int bricked;    // 0: x-fastest;  1: 8^3 bricks (x-fastest over bricks), Morton order inside;
                  // 2: bm^3 bricks (x-fastest over bricks), x-fastest inside (the cells of a macro cube)
  int nbk;        // bricks per axis (bricked)
  int bm;         // brick edge (bricked = 2)
};
__host__ __device__ __forceinline__ unsigned dil3(unsigned v) {      // 3 bits -> every third bit
  return (v & 1u) | ((v & 2u) << 2) | ((v & 4u) << 4);
}
__host__ __device__ __forceinline__ unsigned undil3(unsigned m) {
  return (m & 1u) | ((m >> 2) & 2u) | ((m >> 4) & 4u);
}
// contribution of coordinate i on axis a to the storage slot
__host__ __device__ __forceinline__ long long axis_term(const LayoutU& L, int a, int i) {
  if (L.bricked == 1) {
    long long bs = a == 0 ? 1 : (a == 1 ? L.nbk : (long long)L.nbk * L.nbk);
    return (long long)(dil3((unsigned)i & 7u) << a) + 512ll * (i >> 3) * bs;
  }
  if (L.bricked == 2) {
    long long bs = a == 0 ? 1 : (a == 1 ? L.nbk : (long long)L.nbk * L.nbk);
    long long is = a == 0 ? 1 : (a == 1 ? L.bm : (long long)L.bm * L.bm);
    return (long long)(i % L.bm) * is + (long long)L.bm * L.bm * L.bm * (i / L.bm) * bs;
  }
  long long s = a == 0 ? 1 : (a == 1 ? L.N : (long long)L.N * L.N);
  return s * i;
}
__host__ __device__ __forceinline__ long long slot_of(const LayoutU& L, int ix, int iy, int iz) {
  return axis_term(L, 0, ix) + axis_term(L, 1, iy) + axis_term(L, 2, iz);
}
__host__ __device__ __forceinline__ long long slots_of(const LayoutU& L) {
  if (L.bricked == 1) return 512ll * L.nbk * L.nbk * L.nbk;
  return (long long)L.N * L.N * L.N;                                  // bricked = 2 needs N = nbk * bm: no padding
}
// storage slot -> x-fastest cell number (R22), or -1 for a padding slot
__host__ __device__ __forceinline__ long long ext_of_slot(const LayoutU& L, long long s) {
  if (!L.bricked) return s;
  if (L.bricked == 2) {
    const long long b3 = (long long)L.bm * L.bm * L.bm;
    long long b = s / b3;
    int m = (int)(s % b3);
    int bx = (int)(b % L.nbk), by = (int)((b / L.nbk) % L.nbk), bz = (int)(b / ((long long)L.nbk * L.nbk));
    int ix = bx * L.bm + m % L.bm, iy = by * L.bm + (m / L.bm) % L.bm, iz = bz * L.bm + m / (L.bm * L.bm);
    return ix + (long long)L.N * (iy + (long long)L.N * iz);
  }
  unsigned m = (unsigned)(s & 511);
  long long b = s >> 9;
  int bx = (int)(b % L.nbk), by = (int)((b / L.nbk) % L.nbk), bz = (int)(b / ((long long)L.nbk * L.nbk));
  int ix = bx * 8 + (int)undil3(m), iy = by * 8 + (int)undil3(m >> 1), iz = bz * 8 + (int)undil3(m >> 2);
  if (ix >= L.N || iy >= L.N || iz >= L.N) return -1;
  return ix + (long long)L.N * (iy + (long long)L.N * iz);
}

constexpr int kLutEscape = INT_MIN;       // root table: the step leaves the grid
constexpr int kLutLeave = INT_MIN + 1;    // sub table: the step leaves the refined root cube
constexpr int kLutRegion = INT_MIN + 2;   // root table of a swept grid: the step crosses a region boundary (the
                                          // delta itself is in the second copy of the tables)
constexpr int kSubStride = 16;            // ints per (axis, direction) row of the sub table (64-byte rows, S <= 8):
                                          // [0..S-1] slot deltas (+-S^a, the last one kLutLeave), [15] = -(S-1) * delta
constexpr int kPending = (int)0x80000000u; // PacketU::cb: the package crossed into a new root cube at the sub level
                                          // and the cube's entry (density or marker) is still on its way

// offset (ints) of the sub table behind the root tables, such that its rows are 64-byte aligned when the
// table block itself is (the kernel places it at a 64-byte aligned shared-memory address)
__host__ __device__ __forceinline__ int lut_sub_offset(int N) { return (6 * N + 15) & ~15; }

struct TransportParamsU {
  TransportParams base;          // rho / tally / trow are in STORAGE order here
  const int* __restrict__ lut;   // [6][N] root slot deltas: (axis, forward) at (2*axis)*N, reversed at
                                 // (2*axis+1)*N; two-level grids: [6][kSubStride] sub-cell rows from lut_sub_offset(N)
  LayoutU lay;
  int quorum;                    // leave the walk loop when fewer lanes than this are walking; 0 = automatic
  // region sweeps (kernel template REGION)
  float4* rec;                            // [packages of the batch][3] state of a suspended package
  unsigned long long* list_out;           // packages suspended in this sweep: (region << 32 | package number) ...
  unsigned int* list_out_count;           // ... and how many
  const unsigned int* count_dev;          // NULL: base.count items; else the number of items of this sweep (device)
  int resume;                             // the items are suspended packages (records), not new package numbers
  int region_cells[3], regions_per_axis[3];
  int lut2;                               // byte offset from the marked tables to the plain ones in shared memory
  int tail;                               // end of a batch: 1 = once the work queue is empty the walk quorum follows the
                                          // number of packages the warp still holds (0: it drops to 1)
  // a9 fused into this launch (cooperative launch; upd_nT = 0: off): behind a grid-wide barrier at the end of the
  // kernel every block updates its share of the leaf temperatures, exactly as k_update_temperature would
  int upd_nT;
  float upd_ln_coef, upd_ln_sub3;
  const float* upd_lnQ;                   // [nT]
  const int* upd_guide;                   // [kGuide]
  const float* upd_lnrho;                 // [slots] ln of the density (k_ln_density)
  float* upd_trow;                        // = base.trow (written here, read-only above)
  long long upd_slots, upd_n3;
  // density staged in shared memory (kernel template DENS = 1 / 2): what every block copies in
  const void* __restrict__ stage;   // DENS 1: the fp32 density array itself; DENS 2: one bit per storage slot
  unsigned stage_bytes;             // multiple of 16
  float pal0, pal1;                 // DENS 2: the two densities (bit 0 / bit 1)
};

// where a kernel instance reads densities from
struct DensU {
  const float* __restrict__ rho;  // DENS 0: global gathers
  uint32_t base;                  // DENS 1, 2: shared-memory byte address of the staged array
  float v0, v1;                   // DENS 2
};
__device__ __forceinline__ uint32_t lds_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
template <int DENS>
__device__ __forceinline__ float density_at(const DensU& D, int slot) {
  if (DENS == 1) return __uint_as_float(lds_u32(D.base + 4u * (uint32_t)slot));
  if (DENS == 2) {
    const uint32_t w = lds_u32(D.base + (((uint32_t)slot >> 3) & ~3u));
    return ((w >> ((uint32_t)slot & 31u)) & 1u) ? D.v1 : D.v0;
  }
  return __ldg(D.rho + slot);
}

// Automatic walk quorum.  A warp that walks until w lanes are left and then spends E instructions on
// one event pass does about L (32 - w) crossings in c L ln(32/w) + E instructions (L = mean crossings
// per flight, c = instructions per step), so the best w grows with L.  Measured optima (profiles/):
// 12-16 at L = 38 (c1); on the two-level disks 17-18 both at L = 160 (c2) and at L = 320 (c3), with a cliff
// below 17 (c2: 16 -> 3.67, 17 -> 3.16, 18 -> 3.13, 20 -> 3.23, 22 -> 3.41 ms; c3: 16 -> 7.60, 18 -> 6.57, 21 -> 6.80):
// w = 14 + 2 log2(L / 24), at least 8 and at most 24 (18 on two-level grids).
// L is taken from the job's own cumulative counters (crossings / flights so far; the first batch
// starts at 16).  A scheduling knob only: results do not depend on it.
__device__ __forceinline__ int auto_quorum(const unsigned long long* __restrict__ counters, int q_max) {
  const float cr = (float)counters[CNT_CROSS], fl = (float)counters[CNT_FLIGHTS];
  if (fl < 1024.f) return 16;
  const int q = 14 + (int)rintf(2.f * log2f(fmaxf(cr / fl, 1.f) * (1.f / 24.f)));
  return min(q_max, max(8, q));
}

// SU_INTERACT_B: interaction found in the second step of a pair -> the cell's density is in the
// alternate register (moved back in the event pass, never inside the walk loop where the move
// would wait for the gather in flight).
enum : int { SU_WALK = 0, SU_INTERACT = 1, SU_ESCAPE = 2, SU_FETCH = 3, SU_DONE = 4, SU_INTERACT_B = 5, SU_SUSPEND = 6 };

struct PacketU {
  float d0, d1, d2;          // direction
  float t0, t1, t2;          // path length (root-cube edges) at which the next leaf face on each axis is met
  float dt0, dt1, dt2;       // 1/|d_a|
  float tcur, tau_rem, rho;  // path length so far in this flight; optical depth left; density here
  uint32_t p0, p1, p2;       // cursors into the delta tables (shared-memory byte addresses)
  int slot;                  // storage slot of the current leaf
  int cb;                    // bin | component << 16 (component: 0 direct, 1 scattered, 2 thermal)
  uint32_t k;                // flight number
  uint32_t off;              // package number within the batch: pid = first + off
  float u1, u2, u3;          // uniforms of the current flight kept for the interaction
  // two-level grids only (dead registers otherwise): state of a package inside a refined cube
  uint32_t r0, r1, r2;       // the root-level cursors while p0..p2 walk the sub table
  int rslot;                 // storage slot of the refined root cube
  int kref;                  // its first leaf slot (what the cube's marker in the root array holds)
  float hs;                  // leaf edge in root-cube edges: 1, or 1/S inside a refined cube
};

__device__ __forceinline__ int lds_s32(uint32_t addr) {
  int v;
  asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}

// direction of a new flight: components too small to ever be the exit axis are nudged (G1)
__device__ __forceinline__ void set_direction(PacketU& p, float a, float b, float c) {
  if (fabsf(a) < 1e-12f) a = copysignf(1e-12f, a);
  if (fabsf(b) < 1e-12f) b = copysignf(1e-12f, b);
  if (fabsf(c) < 1e-12f) c = copysignf(1e-12f, c);
  p.d0 = a; p.d1 = b; p.d2 = c;
  p.dt0 = __frcp_rn(fabsf(a)); p.dt1 = __frcp_rn(fabsf(b)); p.dt2 = __frcp_rn(fabsf(c));
  p.tcur = 0.f;
}
// root-table cursors of root cube (ix,iy,iz) for the current direction (reversed table: entry N-1-i)
__device__ __forceinline__ void root_cursors(const PacketU& p, uint32_t lut, int N, int ix, int iy, int iz,
                                             uint32_t& c0, uint32_t& c1, uint32_t& c2) {
  c0 = lut + 4u * (uint32_t)(p.d0 > 0.f ? ix : 2 * N - 1 - ix);
  c1 = lut + 4u * (uint32_t)(2 * N + (p.d1 > 0.f ? iy : 2 * N - 1 - iy));
  c2 = lut + 4u * (uint32_t)(4 * N + (p.d2 > 0.f ? iz : 2 * N - 1 - iz));
}
// root cube back from root-table cursors
__device__ __forceinline__ void cell_of(const PacketU& p, uint32_t c0, uint32_t c1, uint32_t c2, uint32_t lut,
                                        int N, int& ix, int& iy, int& iz) {
  int q0 = (int)((c0 - lut) >> 2), q1 = (int)((c1 - lut) >> 2) - 2 * N, q2 = (int)((c2 - lut) >> 2) - 4 * N;
  ix = p.d0 > 0.f ? q0 : 2 * N - 1 - q0;
  iy = p.d1 > 0.f ? q1 : 2 * N - 1 - q1;
  iz = p.d2 > 0.f ? q2 : 2 * N - 1 - q2;
}
// Start a flight at the root level: the package sits in root cube (ix,iy,iz) at cube-local
// position (ux,uy,uz) in [0,1]^3; direction already set.
__device__ __forceinline__ void begin_flight(PacketU& p, uint32_t lut, int N, int ix, int iy, int iz,
                                             float ux, float uy, float uz) {
  p.t0 = (p.d0 > 0.f ? 1.f - ux : ux) * p.dt0;
  p.t1 = (p.d1 > 0.f ? 1.f - uy : uy) * p.dt1;
  p.t2 = (p.d2 > 0.f ? 1.f - uz : uz) * p.dt2;
  root_cursors(p, lut, N, ix, iy, iz, p.p0, p.p1, p.p2);
  p.hs = 1.f;
}
// sub-table cursor of (axis, direction sign, directional index j = number of subcubes behind)
__device__ __forceinline__ uint32_t sub_cursor(uint32_t sublut, int axis, float d, int j) {
  return sublut + 4u * (uint32_t)((2 * axis + (d > 0.f ? 0 : 1)) * kSubStride + j);
}
// Start a flight inside subcube (sx,sy,sz) of the refined root cube (ix,iy,iz) at subcube-local
// position (fx,fy,fz) in [0,1]^3; direction already set; p.slot / p.rslot are the caller's.
__device__ __forceinline__ void begin_flight_sub(PacketU& p, uint32_t lut, uint32_t sublut, int N, int S,
                                                 int ix, int iy, int iz, int sx, int sy, int sz,
                                                 float fx, float fy, float fz) {
  const float hs = 1.f / (float)S;
  p.t0 = (p.d0 > 0.f ? 1.f - fx : fx) * hs * p.dt0;
  p.t1 = (p.d1 > 0.f ? 1.f - fy : fy) * hs * p.dt1;
  p.t2 = (p.d2 > 0.f ? 1.f - fz : fz) * hs * p.dt2;
  root_cursors(p, lut, N, ix, iy, iz, p.r0, p.r1, p.r2);
  p.p0 = sub_cursor(sublut, 0, p.d0, p.d0 > 0.f ? sx : S - 1 - sx);
  p.p1 = sub_cursor(sublut, 1, p.d1, p.d1 > 0.f ? sy : S - 1 - sy);
  p.p2 = sub_cursor(sublut, 2, p.d2, p.d2 > 0.f ? sz : S - 1 - sz);
  p.hs = hs;
}
// directional subcube index on one axis from a sub-table cursor (rows are 64-byte aligned)
__device__ __forceinline__ int sub_j(uint32_t cursor) {
  return (int)((cursor >> 2) & (uint32_t)(kSubStride - 1));
}

// A package at the root level whose gathered "density" is the marker of a refined cube (sign bit
// | storage slot of its first subcube): descend into the subcube it is in.  Per axis the remaining distance to
// the cube's exit face, in subcube edges, W = (t_a - tcur)|d_a| S, selects the subcube: m =
// ceil(W) - 1 whole subcubes lie between the package's subcube and that face (a package exactly on
// a subcube face belongs to the subcube it flies into: direction-aware as R7; the entry axis has
// W = S).  Then t_a shrinks to the subcube's own exit face and the cursors move to the sub table.
__device__ __forceinline__ void descend(const TransportParams& P, PacketU& p, uint32_t sublut, float& cur) {
  const int S = P.S;
  const float fS = (float)S, hs = 1.f / fS;
  const int kref = __float_as_int(cur) & 0x7fffffff;        // first leaf slot of the refined cube
  const int m0 = min(S - 1, max(0, (int)ceilf((p.t0 - p.tcur) * fabsf(p.d0) * fS) - 1));
  const int m1 = min(S - 1, max(0, (int)ceilf((p.t1 - p.tcur) * fabsf(p.d1) * fS) - 1));
  const int m2 = min(S - 1, max(0, (int)ceilf((p.t2 - p.tcur) * fabsf(p.d2) * fS) - 1));
  p.t0 = fmaxf(p.tcur, p.t0 - (float)m0 * hs * p.dt0);
  p.t1 = fmaxf(p.tcur, p.t1 - (float)m1 * hs * p.dt1);
  p.t2 = fmaxf(p.tcur, p.t2 - (float)m2 * hs * p.dt2);
  p.r0 = p.p0; p.r1 = p.p1; p.r2 = p.p2;
  p.rslot = p.slot;
  const int j0 = S - 1 - m0, j1 = S - 1 - m1, j2 = S - 1 - m2;
  p.p0 = sub_cursor(sublut, 0, p.d0, j0);
  p.p1 = sub_cursor(sublut, 1, p.d1, j1);
  p.p2 = sub_cursor(sublut, 2, p.d2, j2);
  const int sx = p.d0 > 0.f ? j0 : m0, sy = p.d1 > 0.f ? j1 : m1, sz = p.d2 > 0.f ? j2 : m2;
  p.slot = kref + sx + S * (sy + S * sz);
  p.kref = kref;
  p.hs = hs;
  MCRT_CHECK_SLOT(p.slot);
  cur = __ldg(P.rho + p.slot);
}

// A package at the sub level whose exits must move out to the faces of its root cube (it has left
// the refined region, or the grid): per axis (S - 1 - j) more subcube edges; cursors back to the
// root tables.  The exit axis of a kLutLeave step has j = 0 by then, so one rule serves all three.
__device__ __forceinline__ void to_root_level(const TransportParams& P, PacketU& p) {
  const int S = P.S;
  const float h = p.hs;
  p.t0 = fmaf((float)(S - 1 - sub_j(p.p0)) * h, p.dt0, p.t0);
  p.t1 = fmaf((float)(S - 1 - sub_j(p.p1)) * h, p.dt1, p.t1);
  p.t2 = fmaf((float)(S - 1 - sub_j(p.p2)) * h, p.dt2, p.t2);
  p.p0 = p.r0; p.p1 = p.r1; p.p2 = p.r2;
  p.slot = p.rslot;
  p.hs = 1.f;
}

// Start of a step on a two-level grid when the gathered entry is a refined-cube marker or the
// package is waiting for the entry of the root cube it crossed into (kPending):
//  * pending + marker: refined -> refined, the leaf slot moves to the same subcube of the new cube
//    (the wrap of the exit axis was applied when the step was taken), then its density is gathered;
//  * pending, no marker: the package has left the refined region -> root level, `cur` is its density;
//  * marker, not pending: a package at the root level meets a refined cube -> descend().
__device__ __forceinline__ void root_entry(const TransportParams& P, PacketU& p, uint32_t sublut, float& cur) {
  const int bits = __float_as_int(cur);
  if (p.cb < 0) {
    p.cb &= ~kPending;
    if (bits < 0) {
      const int kref = bits & 0x7fffffff;
      p.slot += kref - p.kref;
      p.kref = kref;
      MCRT_CHECK_SLOT(p.slot);
      cur = __ldg(P.rho + p.slot);
    } else {
      to_root_level(P, p);
    }
  } else {
    descend(P, p, sublut, cur);
  }
}

// One crossing of the cell walk (O5).  `cur` holds the density of the current leaf; the density
// of the next leaf is requested into `nxt` BEFORE the optical-depth test, so consecutive calls
// alternate the two registers and no instruction waits on the gather except its real use.
// tau_rem > 0 always (u01 < 1, and a - b > 0 for a > b in IEEE arithmetic), so dtau >= tau_rem
// implies rho*kappa > 0: no interaction in an empty leaf (R14).
template <bool TL, int DENS, bool MACRO, bool REGION, int INTERACT = SU_INTERACT>
__device__ __forceinline__ void walk_step_u(const TransportParams& P, const DensU& D, PacketU& p, float& cur,
                                            float& nxt, float kx, uint32_t sublut, int& state, uint32_t& crossings) {
  if (TL) {
    if ((p.cb | __float_as_int(cur)) < 0) root_entry(P, p, sublut, cur);
  }
  const float tnext = fminf(p.t0, fminf(p.t1, p.t2));
  const bool a0 = p.t0 == tnext;                             // ties -> lowest axis (R21)
  const bool a1 = !a0 && p.t1 == tnext;
  const uint32_t csel = a0 ? p.p0 : (a1 ? p.p1 : p.p2);
  int dl = lds_s32(csel);
  int from = p.slot;
  bool leave = false;
  bool cross = false;                                        // REGION: the step crosses a region boundary
  if (REGION) {
    cross = dl == kLutRegion;
    if (cross) dl = lds_s32(csel + sublut);                  // (sublut = offset to the plain tables here)
  }
  if (TL) {
    leave = dl == kLutLeave;
    if (leave) {                                             // the step leaves the refined cube: root table
      dl = lds_s32(a0 ? p.r0 : (a1 ? p.r1 : p.r2));
      from = p.rslot;
    }
  }
  const bool esc = dl == kLutEscape;
  const int nslot = from + dl;
  if (!esc && !(REGION && cross)) { MCRT_CHECK_SLOT(nslot); nxt = density_at<DENS>(D, nslot); }
  const float dtau = cur * kx * (tnext - p.tcur);
  if (dtau >= p.tau_rem) {                                   // interaction inside this leaf
    state = INTERACT;
  } else {
    p.tau_rem -= dtau;
    p.tcur = tnext;
    if (TL && !MACRO) ++crossings;                           // MACRO: counted from the ends of the flight; single-level
                                                             // grids: from the table cursors at the ends of the flight
    if (TL) {
      uint32_t cnew = csel + 4u;
      if (leave) {
        // Keep walking at the sub level: the subcube index of the exit axis wraps (cursor back to the
        // row's start, leaf slot to the mirror subcube), the root cursor of that axis advances, and
        // the entry of the new root cube (density or marker) arrives with the next step (kPending).
        cnew = csel & ~63u;
        p.slot += lds_s32(cnew + 4u * (uint32_t)(kSubStride - 1));
        p.rslot = nslot;
        p.r0 = a0 ? p.r0 + 4u : p.r0; p.r1 = a1 ? p.r1 + 4u : p.r1; p.r2 = (!a0 && !a1) ? p.r2 + 4u : p.r2;
        p.cb |= kPending;
      } else {
        p.slot = nslot;
      }
      const bool a2 = !a0 && !a1;
      p.t0 = a0 ? fmaf(p.dt0, p.hs, p.t0) : p.t0; p.p0 = a0 ? cnew : p.p0;
      p.t1 = a1 ? fmaf(p.dt1, p.hs, p.t1) : p.t1; p.p1 = a1 ? cnew : p.p1;
      p.t2 = a2 ? fmaf(p.dt2, p.hs, p.t2) : p.t2; p.p2 = a2 ? cnew : p.p2;
      if (esc) {
        if (leave) { p.cb &= ~kPending; to_root_level(P, p); }   // left the grid from a subcube (rare)
        state = SU_ESCAPE;
      }
    } else {
      const bool a2 = !a0 && !a1;
      p.t0 = a0 ? p.t0 + p.dt0 : p.t0; p.p0 = a0 ? p.p0 + 4u : p.p0;
      p.t1 = a1 ? p.t1 + p.dt1 : p.t1; p.p1 = a1 ? p.p1 + 4u : p.p1;
      p.t2 = a2 ? p.t2 + p.dt2 : p.t2; p.p2 = a2 ? p.p2 + 4u : p.p2;
      p.slot = nslot;
      if (esc) state = SU_ESCAPE;
      else if (REGION && cross) state = SU_SUSPEND;          // it now sits in the first cell of the next region
    }
  }
}

// The same two steps for single-level grids with global gathers, written in PTX as ONE block: the axis update stays
// predicated, nothing is recomputed, and a package that stops in the first step leaves without a second test.
// Same operations in the same order as walk_step_u (so the results are bit-identical; the checked build keeps the
// C++ form).  States: 1 = SU_INTERACT, 5 = SU_INTERACT_B (the leaf's density is in the second register), 2 =
// SU_ESCAPE, 6 = SU_SUSPEND; table marks: INT_MIN = kLutEscape, INT_MIN + 2 = kLutRegion.
static_assert(SU_WALK == 0 && SU_INTERACT == 1 && SU_ESCAPE == 2 && SU_INTERACT_B == 5 && SU_SUSPEND == 6, "walk_pair_ptx");
static_assert(kLutEscape == -2147483647 - 1 && kLutRegion == -2147483646, "walk_pair_ptx");
template <bool REGION>
__device__ __forceinline__ void walk_pair_ptx(const float* __restrict__ rho, PacketU& p, float& rho_a, float& rho_b,
                                              const float kx, const uint32_t lut2, int& state) {
  if (REGION) {
    asm volatile(
        "{\n"
        ".reg .pred a0, a01, na0, a1, ne, hit, rg, ldp, stop;\n"
        ".reg .f32 tn, ds, s, dtau;\n"
        ".reg .u32 c, c2;\n"
        ".reg .s32 dl, ns;\n"
        ".reg .u64 ad;\n"
        "min.f32 tn, %1, %2;\n"
        "min.f32 tn, %0, tn;\n"
        "setp.eq.f32 a0, %0, tn;\n"
        "setp.eq.or.f32 a01, %1, tn, a0;\n"
        "selp.u32 c, %5, %6, a0;\n"
        "selp.u32 c, c, %7, a01;\n"
        "ld.shared.s32 dl, [c];\n"
        "setp.eq.s32 rg, dl, -2147483646;\n"
        "add.u32 c2, c, %17;\n"
        "@rg ld.shared.s32 dl, [c2];\n"
        "setp.ne.s32 ne, dl, -2147483648;\n"
        "add.s32 ns, %8, dl;\n"
        "mul.wide.s32 ad, ns, 4;\n"
        "add.u64 ad, ad, %16;\n"
        "and.pred ldp, ne, !rg;\n"
        "@ldp ld.global.nc.f32 %11, [ad];\n"
        "sub.f32 ds, tn, %3;\n"
        "mul.f32 s, %10, %15;\n"
        "mul.f32 dtau, s, ds;\n"
        "setp.ge.f32 hit, dtau, %4;\n"
        "@hit mov.s32 %9, 1;\n"
        "@hit bra MCRT_PAIR_DONE;\n"
        "sub.f32 %4, %4, dtau;\n"
        "mov.f32 %3, tn;\n"
        "mov.s32 %8, ns;\n"
        "not.pred na0, a0;\n"
        "and.pred a1, a01, na0;\n"
        "@a0 add.f32 %0, %0, %12;\n"
        "@a0 add.u32 %5, %5, 4;\n"
        "@a1 add.f32 %1, %1, %13;\n"
        "@a1 add.u32 %6, %6, 4;\n"
        "@!a01 add.f32 %2, %2, %14;\n"
        "@!a01 add.u32 %7, %7, 4;\n"
        "@rg mov.s32 %9, 6;\n"
        "@!ne mov.s32 %9, 2;\n"
        "or.pred stop, rg, !ne;\n"
        "@stop bra MCRT_PAIR_DONE;\n"
        "min.f32 tn, %1, %2;\n"
        "min.f32 tn, %0, tn;\n"
        "setp.eq.f32 a0, %0, tn;\n"
        "setp.eq.or.f32 a01, %1, tn, a0;\n"
        "selp.u32 c, %5, %6, a0;\n"
        "selp.u32 c, c, %7, a01;\n"
        "ld.shared.s32 dl, [c];\n"
        "setp.eq.s32 rg, dl, -2147483646;\n"
        "add.u32 c2, c, %17;\n"
        "@rg ld.shared.s32 dl, [c2];\n"
        "setp.ne.s32 ne, dl, -2147483648;\n"
        "add.s32 ns, %8, dl;\n"
        "mul.wide.s32 ad, ns, 4;\n"
        "add.u64 ad, ad, %16;\n"
        "and.pred ldp, ne, !rg;\n"
        "@ldp ld.global.nc.f32 %10, [ad];\n"
        "sub.f32 ds, tn, %3;\n"
        "mul.f32 s, %11, %15;\n"
        "mul.f32 dtau, s, ds;\n"
        "setp.ge.f32 hit, dtau, %4;\n"
        "@hit mov.s32 %9, 5;\n"
        "@hit bra MCRT_PAIR_DONE;\n"
        "sub.f32 %4, %4, dtau;\n"
        "mov.f32 %3, tn;\n"
        "mov.s32 %8, ns;\n"
        "not.pred na0, a0;\n"
        "and.pred a1, a01, na0;\n"
        "@a0 add.f32 %0, %0, %12;\n"
        "@a0 add.u32 %5, %5, 4;\n"
        "@a1 add.f32 %1, %1, %13;\n"
        "@a1 add.u32 %6, %6, 4;\n"
        "@!a01 add.f32 %2, %2, %14;\n"
        "@!a01 add.u32 %7, %7, 4;\n"
        "@rg mov.s32 %9, 6;\n"
        "@!ne mov.s32 %9, 2;\n"
        "MCRT_PAIR_DONE:\n"
        "}\n"
        : "+f"(p.t0), "+f"(p.t1), "+f"(p.t2), "+f"(p.tcur), "+f"(p.tau_rem), "+r"(p.p0), "+r"(p.p1), "+r"(p.p2),
          "+r"(p.slot), "+r"(state), "+f"(rho_a), "+f"(rho_b)
        : "f"(p.dt0), "f"(p.dt1), "f"(p.dt2), "f"(kx), "l"(rho), "r"(lut2)
        : "memory");
  } else {
    asm volatile(
        "{\n"
        ".reg .pred a0, a01, na0, a1, ne, hit, rg, ldp, stop;\n"
        ".reg .f32 tn, ds, s, dtau;\n"
        ".reg .u32 c, c2;\n"
        ".reg .s32 dl, ns;\n"
        ".reg .u64 ad;\n"
        "min.f32 tn, %1, %2;\n"
        "min.f32 tn, %0, tn;\n"
        "setp.eq.f32 a0, %0, tn;\n"
        "setp.eq.or.f32 a01, %1, tn, a0;\n"
        "selp.u32 c, %5, %6, a0;\n"
        "selp.u32 c, c, %7, a01;\n"
        "ld.shared.s32 dl, [c];\n"
        "setp.ne.s32 ne, dl, -2147483648;\n"
        "add.s32 ns, %8, dl;\n"
        "mul.wide.s32 ad, ns, 4;\n"
        "add.u64 ad, ad, %16;\n"
        "@ne ld.global.nc.f32 %11, [ad];\n"
        "sub.f32 ds, tn, %3;\n"
        "mul.f32 s, %10, %15;\n"
        "mul.f32 dtau, s, ds;\n"
        "setp.ge.f32 hit, dtau, %4;\n"
        "@hit mov.s32 %9, 1;\n"
        "@hit bra MCRT_PAIR_DONE;\n"
        "sub.f32 %4, %4, dtau;\n"
        "mov.f32 %3, tn;\n"
        "mov.s32 %8, ns;\n"
        "not.pred na0, a0;\n"
        "and.pred a1, a01, na0;\n"
        "@a0 add.f32 %0, %0, %12;\n"
        "@a0 add.u32 %5, %5, 4;\n"
        "@a1 add.f32 %1, %1, %13;\n"
        "@a1 add.u32 %6, %6, 4;\n"
        "@!a01 add.f32 %2, %2, %14;\n"
        "@!a01 add.u32 %7, %7, 4;\n"
        "@!ne mov.s32 %9, 2;\n"
        "@!ne bra MCRT_PAIR_DONE;\n"
        "min.f32 tn, %1, %2;\n"
        "min.f32 tn, %0, tn;\n"
        "setp.eq.f32 a0, %0, tn;\n"
        "setp.eq.or.f32 a01, %1, tn, a0;\n"
        "selp.u32 c, %5, %6, a0;\n"
        "selp.u32 c, c, %7, a01;\n"
        "ld.shared.s32 dl, [c];\n"
        "setp.ne.s32 ne, dl, -2147483648;\n"
        "add.s32 ns, %8, dl;\n"
        "mul.wide.s32 ad, ns, 4;\n"
        "add.u64 ad, ad, %16;\n"
        "@ne ld.global.nc.f32 %10, [ad];\n"
        "sub.f32 ds, tn, %3;\n"
        "mul.f32 s, %11, %15;\n"
        "mul.f32 dtau, s, ds;\n"
        "setp.ge.f32 hit, dtau, %4;\n"
        "@hit mov.s32 %9, 5;\n"
        "@hit bra MCRT_PAIR_DONE;\n"
        "sub.f32 %4, %4, dtau;\n"
        "mov.f32 %3, tn;\n"
        "mov.s32 %8, ns;\n"
        "not.pred na0, a0;\n"
        "and.pred a1, a01, na0;\n"
        "@a0 add.f32 %0, %0, %12;\n"
        "@a0 add.u32 %5, %5, 4;\n"
        "@a1 add.f32 %1, %1, %13;\n"
        "@a1 add.u32 %6, %6, 4;\n"
        "@!a01 add.f32 %2, %2, %14;\n"
        "@!a01 add.u32 %7, %7, 4;\n"
        "@!ne mov.s32 %9, 2;\n"
        "MCRT_PAIR_DONE:\n"
        "}\n"
        : "+f"(p.t0), "+f"(p.t1), "+f"(p.t2), "+f"(p.tcur), "+f"(p.tau_rem), "+r"(p.p0), "+r"(p.p1), "+r"(p.p2),
          "+r"(p.slot), "+r"(state), "+f"(rho_a), "+f"(rho_b)
        : "f"(p.dt0), "f"(p.dt1), "f"(p.dt2), "f"(kx), "l"(rho), "r"(lut2)
        : "memory");
  }
}

// O4: where a new package starts.  Point source: finest-level cell fx.. and fractional position
// in it (direction-aware on a face, R7).  External field (R25): a point on one of the six box
// faces and an inward cosine-law direction; returns the ROOT cube and cube-local position.
// r = float uniforms of the Philox block (pid, 0, EMIT).
__device__ __forceinline__ void emit_position_u(const TransportParams& P, const SrcDev& sd,
                                                unsigned long long pid, const float r[4], int& ix,
                                                int& iy, int& iz, float& ux, float& uy, float& uz,
                                                float& a, float& b, float& c) {
  const int N = P.N;
  if (sd.type == 0) {
    ix = sd.fine[0]; iy = sd.fine[1]; iz = sd.fine[2];
    ux = sd.frac[0]; uy = sd.frac[1]; uz = sd.frac[2];
    if (a < 0.f && ux == 0.f) { --ix; ux = 1.f; }             // R7: ceil(x) - 1 for d < 0
    if (b < 0.f && uy == 0.f) { --iy; uy = 1.f; }
    if (c < 0.f && uz == 0.f) { --iz; uz = 1.f; }
  } else {                                                    // R25 external isotropic field
    float v[4];
    draw4(P.seed, pid, 1, kTagEmit, v);
    int f = min(5, (int)(6.f * v[0]));
    int ax = f >> 1, side = f & 1;
    float mu = sqrtf(r[2]);
    float st = sqrtf(fmaxf(0.f, 1.f - mu * mu));
    float sn, cs;
    sincospif(2.f * r[3], &sn, &cs);
    float dn = side == 0 ? mu : -mu, e1 = st * cs, e2 = st * sn;     // normal, axis+1, axis+2
    float fN = (float)N;
    float x1 = v[1] * fN, x2 = v[2] * fN;
    int i1 = min(N - 1, (int)x1), i2 = min(N - 1, (int)x2);
    float l1 = x1 - (float)i1, l2 = x2 - (float)i2;
    if (e1 < 0.f && l1 == 0.f && i1 > 0) { --i1; l1 = 1.f; }
    if (e2 < 0.f && l2 == 0.f && i2 > 0) { --i2; l2 = 1.f; }
    int in = side == 0 ? 0 : N - 1;
    float ln = side == 0 ? 0.f : 1.f;
    if (ax == 0)      { a = dn; b = e1; c = e2; ix = in; iy = i1; iz = i2; ux = ln; uy = l1; uz = l2; }
    else if (ax == 1) { a = e2; b = dn; c = e1; iy = in; iz = i1; ix = i2; uy = ln; uz = l1; ux = l2; }
    else              { a = e1; b = e2; c = dn; iz = in; ix = i1; iy = i2; uz = ln; ux = l1; uy = l2; }
  }
}

// MINBLOCKS = resident blocks per SM the kernel is compiled for: 4 (64 registers) or 5 (48
// registers).  Five blocks hide more of the L2 latency on cache-resident grids; on HBM-resident
// grids the extra threads thrash the L1, so the host picks per grid (profiles/).
// signed sum of the cell coordinates along the direction of flight: a flight from cell F to cell F' crosses
// sum_a sign(d_a) (F'_a - F_a) cell faces (per axis the motion is monotonic)
__device__ __forceinline__ uint32_t along(const PacketU& p, int f0, int f1, int f2) {
  return (uint32_t)((p.d0 > 0.f ? f0 : -f0) + (p.d1 > 0.f ? f1 : -f1) + (p.d2 > 0.f ? f2 : -f2));
}

// Single-level grids: every crossing moves exactly one of the three table cursors on by one entry, so the crossings
// of a flight are the difference of this sum between its end and its start (R27; no counter in the walk loop).
__device__ __forceinline__ uint32_t cursor_sum(const PacketU& p) { return (p.p0 + p.p1 + p.p2) >> 2; }

// PAH: the instance that knows the transiently heated PAH (row f2).  A template parameter, not a run-time
// branch: the third Philox block in the event pass costs registers and spills in every instance that
// contains it (C2 3.38 -> 3.52 ms per launch when it was compiled into all of them).
template <int MINBLOCKS, bool TL, int DENS, bool MACRO, bool PAH, bool REGION>
__global__ void __launch_bounds__(256, MINBLOCKS) k_transport_u(const TransportParamsU PU) {
  const TransportParams& P = PU.base;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float4* s_opac = reinterpret_cast<float4*>(smem_raw);                    // [nb]
  uint32_t* s_sed = reinterpret_cast<uint32_t*>(s_opac + P.nb);             // [3*nb]
  uint32_t* s_emit = s_sed + 3 * P.nb;                                      // [nb]
  // root delta tables [6*N] (+ the 64-byte aligned sub-table rows), at a 64-byte aligned address
  int* s_lut = reinterpret_cast<int*>(smem_raw + ((32u * (unsigned)P.nb + 63u) & ~63u));
  const uint32_t lut = (uint32_t)__cvta_generic_to_shared(s_lut);
  const int N = P.N;
  // two-level grids: address of the subcube rows; swept grids: byte OFFSET from the marked to the plain root tables
  const uint32_t sublut = REGION ? 4u * (uint32_t)(6 * N) : lut + 4u * (uint32_t)lut_sub_offset(N);
  const int n_lut = TL ? lut_sub_offset(N) + 6 * kSubStride : (REGION ? 12 * N : 6 * N);
  const unsigned long long n_items = REGION && PU.count_dev ? (unsigned long long)*PU.count_dev : P.count;
  for (int i = threadIdx.x; i < P.nb; i += blockDim.x) { s_opac[i] = P.opac[i]; s_emit[i] = 0; }
  for (int i = threadIdx.x; i < 3 * P.nb; i += blockDim.x) s_sed[i] = 0;
  for (int i = threadIdx.x; i < n_lut; i += blockDim.x) s_lut[i] = PU.lut[i];
  if (blockIdx.x == 0 && threadIdx.x == 0) *P.next_reset = 0ull;
  DensU D;
  D.rho = P.rho; D.base = 0; D.v0 = PU.pal0; D.v1 = PU.pal1;
  if (DENS != 0) {
    // the staged density array behind the tables (128-byte aligned), then the mbarrier of its bulk copy
    const uint32_t off = (uint32_t)(((32u * (unsigned)P.nb + 63u) & ~63u) + 4u * (unsigned)n_lut + 127u) & ~127u;
    D.base = (uint32_t)__cvta_generic_to_shared(smem_raw) + off;
    const uint32_t bar = D.base + PU.stage_bytes;
    if (threadIdx.x == 0) {
      asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar));
      asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(PU.stage_bytes) : "memory");
      asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                   ::"r"(D.base), "l"(PU.stage), "r"(PU.stage_bytes), "r"(bar) : "memory");
    }
    __syncthreads();                                         // the barrier is initialised for everyone
    asm volatile("{\n.reg .pred p;\nMCRT_STAGE_WAIT:\n"
                 "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], 0;\n"
                 "@p bra MCRT_STAGE_DONE;\nbra MCRT_STAGE_WAIT;\nMCRT_STAGE_DONE:\n}" ::"r"(bar) : "memory");
  }
  __syncthreads();

  const unsigned lane = threadIdx.x & 31;
  const unsigned lt_mask = (1u << lane) - 1u;
  // event counters kept per lane: crossings, absorptions, scatterings, flights.  Emitted and
  // escaped packages are counted by the block's emission / SED histograms (summed at the end),
  // lost packages (R20, must never happen) go straight to the global counter.
  uint32_t n_cross = 0, n_abs = 0, n_sca = 0, n_flights = 0;

  PacketU p;
  p.d0 = p.d1 = p.d2 = 1.f; p.t0 = p.t1 = p.t2 = 0.f; p.dt0 = p.dt1 = p.dt2 = 1.f;
  p.tcur = 0.f; p.tau_rem = 1.f; p.rho = 0.f; p.p0 = p.p1 = p.p2 = lut; p.slot = 0;
  p.r0 = p.r1 = p.r2 = lut; p.rslot = 0; p.kref = 0; p.hs = 1.f;
  float rho_b = 0.f;                                         // the walk alternates p.rho / rho_b
  p.cb = 0; p.k = 0; p.off = 0; p.u1 = p.u2 = p.u3 = 0.f;
  float kx = 0.f;
  int state = SU_FETCH;
  const int quorum0 = PU.quorum > 0 ? PU.quorum : auto_quorum(P.counters, TL && !MACRO ? 18 : 24);
  int quorum = quorum0;
  bool tail = false;                                         // the work queue is (nearly) empty

  for (;;) {
    // ---- a7: escaped packages -> SED; a8: refill from the work queue (one atomic per warp) ----
    if (state == SU_ESCAPE) {
      if (!TL) n_cross += cursor_sum(p);
      if (MACRO || (P.obs.n_mu | P.obs.n_pix)) {             // exit point: cube from the cursors, offset from the t's
        int ix, iy, iz;                                      // (a package always leaves the grid at the root level)
        cell_of(p, p.p0, p.p1, p.p2, lut, N, ix, iy, iz);
        const float w0 = fminf(1.f, fmaxf(0.f, (p.t0 - p.tcur) * fabsf(p.d0)));
        const float w1 = fminf(1.f, fmaxf(0.f, (p.t1 - p.tcur) * fabsf(p.d1)));
        const float w2 = fminf(1.f, fmaxf(0.f, (p.t2 - p.tcur) * fabsf(p.d2)));
        const float ex = p.d0 > 0.f ? 1.f - w0 : w0, ey = p.d1 > 0.f ? 1.f - w1 : w1, ez = p.d2 > 0.f ? 1.f - w2 : w2;
        if (MACRO) {                                         // cell coordinates where the flight ends: beyond the box on the exit axis
          const int S = P.S;
          const int f0 = ix >= N ? N * S : (ix < 0 ? -1 : ix * S + min(S - 1, (int)(ex * (float)S)));
          const int f1 = iy >= N ? N * S : (iy < 0 ? -1 : iy * S + min(S - 1, (int)(ey * (float)S)));
          const int f2 = iz >= N ? N * S : (iz < 0 ? -1 : iz * S + min(S - 1, (int)(ez * (float)S)));
          n_cross += along(p, f0, f1, f2);
        }
        if (P.obs.n_mu | P.obs.n_pix)
          tally_observer(P, (float)ix + ex, (float)iy + ey, (float)iz + ez, p.d0, p.d1, p.d2, p.cb & 0xffff, p.cb >> 16);
      }
      atomicAdd(&s_sed[(p.cb >> 16) * P.nb + (p.cb & 0xffff)], 1u);
      state = SU_FETCH;
    }
    if (REGION) {                                            // packages that crossed into another region wait for its sweep
      const unsigned sm = __ballot_sync(kFull, state == SU_SUSPEND);
      if (state == SU_SUSPEND) {
        int ix, iy, iz;
        n_cross += cursor_sum(p);
        cell_of(p, p.p0, p.p1, p.p2, lut, N, ix, iy, iz);
        const unsigned key = (unsigned)(ix / PU.region_cells[0] + PU.regions_per_axis[0] *
                                        (iy / PU.region_cells[1] + PU.regions_per_axis[1] * (iz / PU.region_cells[2])));
        float4* r = PU.rec + 3 * (size_t)p.off;
        r[0] = make_float4(p.d0, p.d1, p.d2, p.tcur);
        r[1] = make_float4(p.t0, p.t1, p.t2, p.tau_rem);
        r[2] = make_float4(__int_as_float(ix | (iy << 16)), __int_as_float(iz), __int_as_float(p.cb),
                           __int_as_float((int)p.k));
        const int leader = __ffs(sm) - 1;
        unsigned base = 0;
        if ((int)lane == leader) base = atomicAdd(PU.list_out_count, (unsigned)__popc(sm));
        base = __shfl_sync(sm, base, leader);
        PU.list_out[base + __popc(sm & lt_mask)] = ((unsigned long long)key << 32) | p.off;
        state = SU_FETCH;
      }
    }
    bool is_new = false;
    const unsigned need = __ballot_sync(kFull, state == SU_FETCH);
    if (need) {
      unsigned long long base = 0;
      if (lane == 0) base = atomicAdd(P.next, (unsigned long long)__popc(need));
      base = __shfl_sync(kFull, base, 0);
      if (base + 32ull > n_items) { quorum = 1; tail = PU.tail != 0; }   // queue (nearly) empty: no more refills
      if (state == SU_FETCH) {
        unsigned long long my = base + (unsigned long long)__popc(need & lt_mask);
        if (my < n_items) {
          p.off = P.perm ? __ldg(P.perm + my) : (uint32_t)my;
          if (REGION && PU.resume) {                         // a suspended package: restore it exactly
            const float4* r = PU.rec + 3 * (size_t)p.off;
            const float4 ra = r[0], rb = r[1], rc = r[2];
            p.d0 = ra.x; p.d1 = ra.y; p.d2 = ra.z; p.tcur = ra.w;
            p.dt0 = __frcp_rn(fabsf(p.d0)); p.dt1 = __frcp_rn(fabsf(p.d1)); p.dt2 = __frcp_rn(fabsf(p.d2));
            p.t0 = rb.x; p.t1 = rb.y; p.t2 = rb.z; p.tau_rem = rb.w;
            const int cxy = __float_as_int(rc.x), ix = cxy & 0xffff, iy = cxy >> 16, iz = __float_as_int(rc.y);
            p.cb = __float_as_int(rc.z); p.k = (uint32_t)__float_as_int(rc.w);
            root_cursors(p, lut, N, ix, iy, iz, p.p0, p.p1, p.p2);
            n_cross -= cursor_sum(p);
            p.slot = (int)slot_of(PU.lay, ix, iy, iz);
            MCRT_CHECK_SLOT(p.slot);
            p.rho = density_at<DENS>(D, p.slot);
            kx = s_opac[p.cb & 0xffff].x;
            float u[4];                                      // the flight's uniforms again (R18: fixed slots)
            draw4(P.seed, P.first + p.off, p.k, kTagFlight, u);
            p.u1 = u[1]; p.u2 = u[2]; p.u3 = u[3];
            state = SU_WALK;
          } else {
            is_new = true;
          }
        } else {
          state = SU_DONE;
        }
      }
    }
    if (__all_sync(kFull, state == SU_DONE)) break;

    // ---- one event pass for every lane that is not walking ----
    if (is_new || state == SU_INTERACT || state == SU_INTERACT_B) {
      if (state == SU_INTERACT_B) p.rho = rho_b;
      const unsigned long long pid = P.first + p.off;
      int bin = p.cb & 0xffff, comp = p.cb >> 16;
      int ix = 0, iy = 0, iz = 0, sx = 0, sy = 0, sz = 0;
      float ux = 0.f, uy = 0.f, uz = 0.f, a, b, c;
      bool scatter = false;
      bool in_sub = TL && !is_new && p.hs < 1.f;             // the package sits in a subcube
      if (!is_new) {                                         // where the interaction happened
        if (!TL) n_cross += cursor_sum(p);
        // it lies tau_rem / (rho kappa) further along this leaf's segment (rho kappa > 0 here)
        const float seg = fminf(p.t0, fminf(p.t1, p.t2)) - p.tcur;
        const float ak = p.rho * kx;
        const float ti = p.tcur + (ak > 0.f ? fminf(seg, p.tau_rem / ak) : 0.f);
        // fraction of the leaf's edge left to its exit face, per axis
        const float ih = in_sub ? (float)P.S : 1.f;
        float w0 = fminf(1.f, fmaxf(0.f, (p.t0 - ti) * fabsf(p.d0) * ih));
        float w1 = fminf(1.f, fmaxf(0.f, (p.t1 - ti) * fabsf(p.d1) * ih));
        float w2 = fminf(1.f, fmaxf(0.f, (p.t2 - ti) * fabsf(p.d2) * ih));
        ux = p.d0 > 0.f ? 1.f - w0 : w0;
        uy = p.d1 > 0.f ? 1.f - w1 : w1;
        uz = p.d2 > 0.f ? 1.f - w2 : w2;
        if (in_sub) {
          cell_of(p, p.r0, p.r1, p.r2, lut, N, ix, iy, iz);
          const int S = P.S, j0 = sub_j(p.p0), j1 = sub_j(p.p1), j2 = sub_j(p.p2);
          sx = p.d0 > 0.f ? j0 : S - 1 - j0;
          sy = p.d1 > 0.f ? j1 : S - 1 - j1;
          sz = p.d2 > 0.f ? j2 : S - 1 - j2;
        } else {
          cell_of(p, p.p0, p.p1, p.p2, lut, N, ix, iy, iz);
          if (MACRO) {                                       // the cell of the uniform macro cube the point lies in
            const int S = P.S;
            sx = min(S - 1, (int)(ux * (float)S)); sy = min(S - 1, (int)(uy * (float)S)); sz = min(S - 1, (int)(uz * (float)S));
          }
        }
        if (MACRO) n_cross += along(p, ix * P.S + sx, iy * P.S + sy, iz * P.S + sz);   // this flight ends here
        scatter = p.u1 < s_opac[bin].y;                      // a4 (R16)
      }
      if (scatter) {                                         // a5
        ++n_sca;
        float ct = hg_cos(s_opac[bin].z, p.u2);
        rotate_dir(p.d0, p.d1, p.d2, ct, p.u3, a, b, c);
        if (comp == 0) comp = 1;
        ++p.k;
      } else {                                               // a1 emission / a6 absorption + re-emission
        uint32_t xw[4];
        draw4w(P.seed, pid, is_new ? 0u : p.k, is_new ? kTagEmit : kTagReemit, xw);
        const float r2 = u01(xw[2]), r3 = u01(xw[3]);
        const float* row;
        float us;
        int s = 0;
        int lo = 0, hi = P.nb - 1;                           // where the bin search starts (narrowed by the rows' guide)
        if (is_new) {                                        // O4: source by luminosity (fp64, exact)
          const double u0 = u01d(xw[0]);
          while (s < P.nsrc - 1 && P.src[s].lcdf < u0) ++s;
          row = P.csrc + (size_t)s * P.nb;
          us = (float)u01d(xw[1]);
        } else {
          ++n_abs;
          int tslot = p.slot;
          if (MACRO && !in_sub) tslot = P.n3 + p.slot * (P.S * P.S * P.S) + sx + P.S * (sy + P.S * sz);
          MCRT_CHECK_SLOT(tslot);
          bool by_pah = false;
          if (PAH) {                                         // R36: which grain took the package
            uint32_t vw[4];
            draw4w(P.seed, pid, p.k, kTagPah, vw);
            by_pah = u01(vw[0]) < __ldg(P.pah_q + bin);
            if (by_pah) {                                    // booked on the leaf's absorbed spectrum; re-emitted
              atomicAdd(P.pah_cnt + (size_t)tslot * P.nb + bin, 1u);      // from the leaf's P(T) (frozen)
              row = P.pah_cdf + (size_t)tslot * P.nb;
              us = u01(vw[1]);
            }
          }
          if (!by_pah) {
            // warp-aggregated integer tally: one atomic per distinct cell per warp
            unsigned peers = __match_any_sync(__activemask(), tslot);
            if ((int)lane == __ffs(peers) - 1) {
              if (P.tally32) atomicAdd(P.tally32 + tslot, (uint32_t)__popc(peers));
              else atomicAdd(P.tally + tslot, (unsigned long long)__popc(peers));
            }
            float tr = __ldg(P.trow + tslot);                // T frozen = T before absorption
            int k0 = min(P.nT - 1, (int)tr);
            float w = tr - (float)k0;
            int rw = (u01(xw[1]) < w && k0 + 1 < P.nT) ? k0 + 1 : k0; // R11 stochastic row choice
            row = P.cdf + (size_t)rw * P.nb;
            us = u01(xw[0]);
            if (P.cdf_guide) {                               // one load instead of the first four or five probes
              const uint32_t g = __ldg(P.cdf_guide + rw * kCdfGuide + (int)(us * (float)kCdfGuide));
              lo = (int)(g & 0xffffu); hi = (int)(g >> 16);
            }
          }
        }
        bin = search_cdf_range<float>(row, lo, hi, us);      // one search loop for emission and re-emission
        if (is_new) {
          // the emission bin is settled in fp64 against the fp64 table with the oracle's uniform: the fp32
          // search lands within a bin or two of "first j with C[j] >= u", a short walk ends exactly on it
          const double* c64 = P.csrc64 + (size_t)s * P.nb;
          const double ud = u01d(xw[1]);
          while (bin > 0 && __ldg(c64 + bin - 1) >= ud) --bin;
          while (bin < P.nb - 1 && __ldg(c64 + bin) < ud) ++bin;
        }
        kx = s_opac[bin].x;
        isotropic_dir(r2, r3, a, b, c);
        if (is_new) {
          const float r[4] = {0.f, 0.f, r2, r3};
          emit_position_u(P, P.src[s], pid, r, ix, iy, iz, ux, uy, uz, a, b, c);
          if (TL && P.src[s].type == 0) {                    // finest-level cell -> root cube + subcube
            const int S = P.S;
            sx = ix % S; sy = iy % S; sz = iz % S;
            ix /= S; iy /= S; iz /= S;
          }
          p.slot = (int)slot_of(PU.lay, ix, iy, iz);
          MCRT_CHECK_SLOT(p.slot);
          p.rho = density_at<DENS>(D, p.slot);
          if (TL && P.src[s].type == 0) {
            if (__float_as_int(p.rho) < 0) {                 // the source sits in a refined cube
              const int S = P.S;
              p.rslot = p.slot;
              p.kref = __float_as_int(p.rho) & 0x7fffffff;
              p.slot = p.kref + sx + S * (sy + S * sz);
              MCRT_CHECK_SLOT(p.slot);
              p.rho = __ldg(P.rho + p.slot);
              in_sub = true;
            } else {                                         // cube-local position from the finest-level one
              const float hs = 1.f / (float)P.S;
              ux = ((float)sx + ux) * hs; uy = ((float)sy + uy) * hs; uz = ((float)sz + uz) * hs;
            }
          } else if (MACRO) {                                // external field: the cell the entry point lies in
            const int S = P.S;
            sx = min(S - 1, (int)(ux * (float)S)); sy = min(S - 1, (int)(uy * (float)S)); sz = min(S - 1, (int)(uz * (float)S));
          }
          comp = 0; p.k = 0;
          atomicAdd(&s_emit[bin], 1u);
        } else {
          comp = 2;
          ++p.k;
        }
      }
      // ---- a2: next flight ----
      p.cb = bin | (comp << 16);
      if (p.k >= kMaxFlights) {                              // R20
        atomicAdd(P.counters + CNT_LOST, 1ull);
        state = SU_FETCH;
      } else {
        set_direction(p, a, b, c);
        if (MACRO) n_cross -= along(p, ix * P.S + sx, iy * P.S + sy, iz * P.S + sz);   // ... and the next one starts here
        if (TL && in_sub) begin_flight_sub(p, lut, sublut, N, P.S, ix, iy, iz, sx, sy, sz, ux, uy, uz);
        else begin_flight(p, lut, N, ix, iy, iz, ux, uy, uz);
        if (!TL) n_cross -= cursor_sum(p);
        float u[4];
        draw4(P.seed, pid, p.k, kTagFlight, u);
        p.tau_rem = -logf(u[0]);
        p.u1 = u[1]; p.u2 = u[2]; p.u3 = u[3];
        ++n_flights;
        state = SU_WALK;
      }
    }

    // End of the batch: without refills the lanes of a warp run dry one by one.  The warp keeps the rhythm of
    // the steady state -- it leaves the walk loop when the share `quorum0 / 32` of the lanes that still walk has
    // stopped -- instead of waiting for its last walker before every event pass.
    if (tail) quorum = max(1, (__popc(__ballot_sync(kFull, state == SU_WALK)) * quorum0) >> 5);

    // ---- a3: cell walk until fewer than `quorum` lanes are walking ----
#pragma unroll 1
    for (;;) {
      // (pairs of steps per ballot: two on swept grids, where flights are long -- c4 32.5 -> 31.5 ms per batch;
      // one elsewhere -- c1_tau1 0.325 -> 0.343 ms with two, c2 / c3 within 1 %)
#pragma unroll
      for (int rep = 0; rep < (REGION ? 2 : 1); ++rep) {
#ifndef MCRT_CHECKS
        if (!TL && DENS == 0) {                              // (compile-time choice)
          if (state == SU_WALK) walk_pair_ptx<REGION>(P.rho, p, p.rho, rho_b, kx, sublut, state);
          continue;
        }
#endif
        if (state == SU_WALK) walk_step_u<TL, DENS, MACRO, REGION>(P, D, p, p.rho, rho_b, kx, sublut, state, n_cross);
        if (state == SU_WALK)
          walk_step_u<TL, DENS, MACRO, REGION, SU_INTERACT_B>(P, D, p, rho_b, p.rho, kx, sublut, state, n_cross);
      }
      if (__popc(__ballot_sync(kFull, state == SU_WALK)) < quorum) break;
    }
  }

  // ---- flush block-private tallies ----
  {
    const int which[4] = {CNT_CROSS, CNT_ABS, CNT_SCA, CNT_FLIGHTS};
    const uint32_t val[4] = {n_cross, n_abs, n_sca, n_flights};
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      unsigned long long v = val[i];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(kFull, v, o);
      if (lane == 0 && v) atomicAdd(P.counters + which[i], v);
    }
  }
  __syncthreads();
  unsigned long long esc = 0, emi = 0;
  for (int i = threadIdx.x; i < 3 * P.nb; i += blockDim.x)
    if (s_sed[i]) { atomicAdd(P.sed + i, (unsigned long long)s_sed[i]); esc += s_sed[i]; }
  for (int i = threadIdx.x; i < P.nb; i += blockDim.x)
    if (s_emit[i]) { atomicAdd(P.emit_bin + i, (unsigned long long)s_emit[i]); emi += s_emit[i]; }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    esc += __shfl_xor_sync(kFull, esc, o);
    emi += __shfl_xor_sync(kFull, emi, o);
  }
  if (lane == 0 && esc) atomicAdd(P.counters + CNT_ESCAPED, esc);
  if (lane == 0 && emi) atomicAdd(P.counters + CNT_EMITTED, emi);

  // ---- a9 in the same launch: when every block has tallied its last absorption (grid-wide barrier; the launch is
  // cooperative, so all blocks are resident), the blocks share the leaves.  Same arithmetic as k_update_temperature
  // (trow_of_leaf), tables read through the L1 instead of shared memory: one launch and its latency less per batch
  // (C0's 10^4-package batches: 0.052 -> 0.048 ms per step; no gain from 2.7e5 leaves on, so the host asks for it on
  // small grids only).
  if (PU.upd_nT) {
    __threadfence();
    cooperative_groups::this_grid().sync();
    const int nT = PU.upd_nT;
    const float lq0 = __ldg(PU.upd_lnQ), lqN = __ldg(PU.upd_lnQ + nT - 1);
    const float inv_w = (float)kGuide / (lqN - lq0);
    const bool use_guide = lq0 > -1e29f && lqN > lq0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < PU.upd_slots; i += stride) {
      const unsigned long long c = __ldcg(P.tally + i);            // (tallied by every block: read from the L2)
      PU.upd_trow[i] = trow_of_leaf(c, __ldg(PU.upd_lnrho + i), i >= PU.upd_n3, PU.upd_ln_coef, PU.upd_ln_sub3, PU.upd_lnQ, PU.upd_guide,
                                    nT, lq0, inv_w, use_guide);
    }
  }
}

// ---- region sweeps: group the suspended packages of a sweep by the region they wait in ----------
// list[i] = region << 32 | package number (i < *n_dev).  Same three steps as the grouped hand-out: histogram,
// exclusive scan, scatter with a per-block reservation (the order inside a region is arbitrary).
__global__ void k_region_hist(const unsigned long long* __restrict__ list, const unsigned int* __restrict__ n_dev,
                              int nreg, unsigned int* __restrict__ counts) {
  extern __shared__ unsigned int s_cnt[];
  for (int i = threadIdx.x; i < nreg; i += blockDim.x) s_cnt[i] = 0;
  __syncthreads();
  const unsigned n = *n_dev;
  for (unsigned i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x)
    atomicAdd(&s_cnt[(unsigned)(list[i] >> 32)], 1u);
  __syncthreads();
  for (int i = threadIdx.x; i < nreg; i += blockDim.x)
    if (s_cnt[i]) atomicAdd(&counts[i], s_cnt[i]);
}
__global__ void k_region_scatter(const unsigned long long* __restrict__ list, const unsigned int* __restrict__ n_dev,
                                 int nreg, unsigned int* __restrict__ cursor, uint32_t* __restrict__ perm) {
  extern __shared__ unsigned int s_cnt[];                    // [2 * nreg]: block histogram, block bases
  for (int i = threadIdx.x; i < 2 * nreg; i += blockDim.x) s_cnt[i] = 0;
  __syncthreads();
  const unsigned n = *n_dev;
  const unsigned per_block = (n + gridDim.x - 1) / gridDim.x;
  const unsigned lo = per_block * blockIdx.x, hi = min(n, lo + per_block);
  for (unsigned i = lo + threadIdx.x; i < hi; i += blockDim.x) atomicAdd(&s_cnt[(unsigned)(list[i] >> 32)], 1u);
  __syncthreads();
  for (int i = threadIdx.x; i < nreg; i += blockDim.x) {
    s_cnt[nreg + i] = s_cnt[i] ? atomicAdd(&cursor[i], s_cnt[i]) : 0u;
    s_cnt[i] = 0;
  }
  __syncthreads();
  for (unsigned i = lo + threadIdx.x; i < hi; i += blockDim.x) {
    const unsigned long long e = list[i];
    const unsigned g = (unsigned)(e >> 32);
    perm[s_cnt[nreg + g] + atomicAdd(&s_cnt[g], 1u)] = (uint32_t)e;
  }
}

// ---- layout conversion (set-up and read-out; storage order never shows at the C ABI, R22) ----
// x-fastest caller densities -> storage order (negative / NaN -> 0; padding slots stay 0)
__global__ void k_encode_uniform(const float* __restrict__ rho_ext, float* __restrict__ rho_store,
                                 LayoutU lay, long long n3) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n3) return;
  int ix = (int)(e % lay.N), iy = (int)((e / lay.N) % lay.N), iz = (int)(e / ((long long)lay.N * lay.N));
  float v = rho_ext[e];
  rho_store[slot_of(lay, ix, iy, iz)] = (v > 0.f) ? v : 0.f;
}
// Two-level grids: root array in storage order; density >= 0, or (sign bit | storage slot of its first subcube)
// for a refined root cube (negative / NaN densities -> 0; padding slots stay 0)
__global__ void k_encode_root(const float* __restrict__ rho_root, const int* __restrict__ refidx,
                              float* __restrict__ out, LayoutU lay, long long n3, long long first_sub, int s3) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n3) return;
  int ix = (int)(e % lay.N), iy = (int)((e / lay.N) % lay.N), iz = (int)(e / ((long long)lay.N * lay.N));
  int k = refidx ? refidx[e] : -1;
  float v = rho_root[e];
  v = (v > 0.f) ? v : 0.f;
  out[slot_of(lay, ix, iy, iz)] = k >= 0 ? __int_as_float((int)(0x80000000u | (unsigned)(first_sub + (long long)k * s3))) : v;
}
// Macro cubes (single-level grids run as two-level ones, see MACRO in the kernel):
// the macro array from the cells stored cube by cube: the common density, or the marker
// (sign bit | storage slot of the cube's first cell) that sends the walk down to the cells.
__global__ void k_macro_entries(const float* __restrict__ cells, float* __restrict__ macro, long long nm3, int m3,
                                long long first_cell) {
  long long m = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (m >= nm3) return;
  const float* c = cells + m * m3;
  const float v0 = c[0];
  bool same = true;
  for (int i = 1; i < m3; ++i) if (c[i] != v0) { same = false; break; }
  macro[m] = same ? v0 : __int_as_float((int)(0x80000000u | (unsigned)(first_cell + m * m3)));
}
// storage order -> x-fastest output
template <typename T>
__global__ void k_store_to_ext(const T* __restrict__ store, T* __restrict__ ext, LayoutU lay, long long n3) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n3) return;
  int ix = (int)(e % lay.N), iy = (int)((e / lay.N) % lay.N), iz = (int)(e / ((long long)lay.N * lay.N));
  ext[e] = store[slot_of(lay, ix, iy, iz)];
}
__global__ void k_trow_to_T_u(const float* __restrict__ trow_store, float* __restrict__ T_ext, LayoutU lay,
                              long long n3, float lnTmin, float dlnT) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n3) return;
  int ix = (int)(e % lay.N), iy = (int)((e / lay.N) % lay.N), iz = (int)(e / ((long long)lay.N * lay.N));
  T_ext[e] = expf(lnTmin + dlnT * trow_store[slot_of(lay, ix, iy, iz)]);
}
// x-fastest tally (sum over ranks, as read out by mcrt_get_cell_energy) -> storage order
__global__ void k_ext_to_store_u64(const unsigned long long* __restrict__ ext, unsigned long long* __restrict__ store,
                                   LayoutU lay, long long n3) {
  long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (e >= n3) return;
  int ix = (int)(e % lay.N), iy = (int)((e / lay.N) % lay.N), iz = (int)(e / ((long long)lay.N * lay.N));
  store[slot_of(lay, ix, iy, iz)] = ext[e];
}

}  // namespace mcrt
