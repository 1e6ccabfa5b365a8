// grpic_lanes.cuh — the fused step over DENSE cell-sorted work items: one contiguous run of particles per lane.
//
// k_step_tiled (grpic_tiled.cuh) walks a work item warp by warp: the 32 lanes of an iteration hold 32 CONSECUTIVE
// particles, which share a cell right after a sort and spread over 5-25 cells a few steps later.  Its deposit therefore
// has to find and resolve address conflicts between lanes in every iteration (match, butterfly, straggler queue):
// 30 % of the instructions and almost half of the stall samples of a config-4 launch (profiles/r2_*).
//
// Here the item is cut the other way, so that lanes never work on neighbouring particles at the same time:
//   - the item's particles are cut into 16-byte blocks (four FP32 / two FP64 particles of one column); kLQuad consecutive
//     lanes share a contiguous region and take its blocks in turn (whole 128-byte lines per warp instruction), each
//     lane's own blocks staying within a region of about two sorted cells;
//   - SoA columns move as 128-bit blocks: cp.async (LDGSTS.128) into a lane-private staging slot of shared memory,
//     updated in place, written back with one LDS.128 + STG.128 per column;
//   - J is accumulated in a lane-PRIVATE window of 3 x 3 cells (4 x 4 nodes x 3 components) in shared memory, laid out
//     [slot][lane] so that a lane's window lives in the lane's own bank: plain conflict-free read-modify-writes,
//     no atomics, no shuffles, no votes, no warp synchronisation anywhere in the particle loop;
//   - the window follows the SORTED cell of the lane's current block (offsets[] of the sort say where each key starts);
//     nodes are addressed modulo 4, so a window that moves by a cell flushes (red.global.add) only the node column that
//     leaves it; a path that leaves the window (drift since the sort) goes to L2 directly;
//   - the field stencil of the tile is staged by TMA and averaged to nodes once per item, as in k_step_tiled.
// The arithmetic of the path (grpic_device.cuh) is the same; only the order of the J additions differs.
// Items too sparse for this to pay (less than `dense_min` particles: windows of one or two particles) stay with
// k_step_tiled; the two kernels split the item table of grpic_sort between them (WorkItem::pad).
#pragma once
#include "grpic_tiled.cuh"

namespace grpic {

// Lanes (= particle runs) per work item and particles per 16-byte block of a real column, by precision.  FP32: 256 lanes,
// two items resident per SM (128 registers); blocks of four.  FP64: 384 lanes, one item per SM (12 warps instead of the
// 8 of k_step_tiled<double>: the FP64 step is bound by dependent-issue latency, so resident warps are what it needs);
// blocks of two, so that a lane's staging slot and window (512 bytes) leave room for them in the 227 KB of the SM.
#ifndef GRPIC_LANES_BLOCK32
#define GRPIC_LANES_BLOCK32 256
#endif
#ifndef GRPIC_LANES_BLOCK64
#define GRPIC_LANES_BLOCK64 384
#endif
template <typename T> constexpr int kLThreads = sizeof(T) == 4 ? GRPIC_LANES_BLOCK32 : GRPIC_LANES_BLOCK64;
template <typename T> constexpr int kLPB = 16 / (int)sizeof(T);      // particles per block
constexpr int kLWin = 3;                       // cells per edge of a lane's private J window
constexpr int kLVals = 3 * 16;                 // slots of a window: [component][4][4] nodes
#ifndef GRPIC_LANES_QUAD
#define GRPIC_LANES_QUAD 8
#endif
constexpr int kLQuad = GRPIC_LANES_QUAD;       // lanes that interleave their 16-byte blocks (8: one 128-byte line)
#ifndef GRPIC_LANES_PREFETCH
#define GRPIC_LANES_PREFETCH 1
#endif
constexpr bool kLPrefetch = GRPIC_LANES_PREFETCH != 0;
static_assert(kLVals * kLThreads<float> >= kRawElems && kLVals * kLThreads<double> >= kRawElems,
              "the raw field stencil is staged in the space of the lane windows");

template <typename T>
constexpr size_t lanes_smem_bytes() {
  // windows + node tile + staged real columns (7 x 16 bytes per lane) + staged cell indices + barrier + sort-key offsets
  return (size_t)(kLVals * kLThreads<T> + kNodeElems<T>) * sizeof(T) + (size_t)kLThreads<T> * (7 * 16 + 2 * 4 * kLPB<T>) + 16 +
         (size_t)(kTile * kTile + 4) * 4;
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(smem_dst)), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

// A lane's window holds the 4 x 4 nodes of 3 x 3 cells.  Node (n1, n2) lives in slot (n1 & 3) * 4 + (n2 & 3) of each
// component ("torus" addressing by absolute node index): when the window moves by one cell only the nodes that leave
// it have to be flushed, nothing is copied, and the slots they leave are the ones the entering nodes use.
// Eight plain read-modify-writes of one deposit segment (layout of deposit_segments) of cell (c1, c2):
template <typename T>
__device__ __forceinline__ void lane_add8(T* pW, int c1, int c2, const T v[8]) {
  constexpr int S = kLThreads<T>;
  const int r0 = (c1 & 3) * 4, r1 = ((c1 + 1) & 3) * 4, q0 = c2 & 3, q1 = (c2 + 1) & 3;
  T* const p00 = pW + (r0 + q0) * S;
  T* const p01 = pW + (r0 + q1) * S;
  T* const p10 = pW + (r1 + q0) * S;
  T* const p11 = pW + (r1 + q1) * S;
  p00[0] += v[0];        p01[0] += v[1];                 // J1(c1+1/2, c2), J1(c1+1/2, c2+1)
  p00[16 * S] += v[2];   p10[16 * S] += v[3];            // J2(c1, c2+1/2), J2(c1+1, c2+1/2)
  p00[32 * S] += v[4];   p10[32 * S] += v[5];            // J3(c1, c2), J3(c1+1, c2)
  p01[32 * S] += v[6];   p11[32 * S] += v[7];            // J3(c1, c2+1), J3(c1+1, c2+1)
}

// The same in two halves, so that the eight loads can be issued ahead of the arithmetic that produces the addends
template <typename T>
struct LaneCell {
  T *p00, *p01, *p10, *p11;
  T o[8];
  __device__ __forceinline__ void load(T* pW, int c1, int c2) {
    constexpr int S = kLThreads<T>;
    const int r0 = (c1 & 3) * 4, r1 = ((c1 + 1) & 3) * 4, q0 = c2 & 3, q1 = (c2 + 1) & 3;
    p00 = pW + (r0 + q0) * S; p01 = pW + (r0 + q1) * S; p10 = pW + (r1 + q0) * S; p11 = pW + (r1 + q1) * S;
    o[0] = p00[0]; o[1] = p01[0]; o[2] = p00[16 * S]; o[3] = p10[16 * S];
    o[4] = p00[32 * S]; o[5] = p10[32 * S]; o[6] = p01[32 * S]; o[7] = p11[32 * S];
  }
  __device__ __forceinline__ void add_store(const T v[8]) const {
    constexpr int S = kLThreads<T>;
    p00[0] = o[0] + v[0]; p01[0] = o[1] + v[1]; p00[16 * S] = o[2] + v[2]; p10[16 * S] = o[3] + v[3];
    p00[32 * S] = o[4] + v[4]; p10[32 * S] = o[5] + v[5]; p01[32 * S] = o[6] + v[6]; p11[32 * S] = o[7] + v[7];
  }
};

// node (n1, n2) of the lane's window: its three non-zero slots go to the J arrays with red.global.add and are zeroed.
// No bounds test: a slot whose node lies outside the arrays is never written (no cell there), so it stays zero.
template <typename T>
__device__ __forceinline__ void lane_flush_node(const Consts<T>& g, const JPtrs<T>& J, T* pW, int n1, int n2) {
  constexpr int S = kLThreads<T>;
  T* const w = pW + (((n1 & 3) * 4) + (n2 & 3)) * S;
  const int64_t a = (int64_t)(n1 + g.ng) * g.ld + (n2 + g.ng);
  const T v0 = w[0], v1 = w[16 * S], v2 = w[32 * S];
  if (v0 != T(0)) { red_add(J.j[0] + a, v0); w[0] = T(0); }
  if (v1 != T(0)) { red_add(J.j[1] + a, v1); w[16 * S] = T(0); }
  if (v2 != T(0)) { red_add(J.j[2] + a, v2); w[32 * S] = T(0); }
}
// the whole window with origin cell (wo1, wo2)
template <typename T>
__device__ __forceinline__ void lane_flush(const Consts<T>& g, const JPtrs<T>& J, T* pW, int wo1, int wo2) {
#pragma unroll 1
  for (int r = 0; r < 4; ++r) {
#pragma unroll
    for (int c = 0; c < 4; ++c) lane_flush_node(g, J, pW, wo1 + r, wo2 + c);
  }
}
// the node column n2 = wo2 that leaves the window when it moves by one cell along x2
template <typename T>
__device__ __forceinline__ void lane_flush_col(const Consts<T>& g, const JPtrs<T>& J, T* pW, int wo1, int wo2) {
#pragma unroll
  for (int r = 0; r < 4; ++r) lane_flush_node(g, J, pW, wo1 + r, wo2);
}

template <typename T, typename CoordT = Coord<T>>
__global__ void __launch_bounds__(kLThreads<T>, (sizeof(T) == 4 ? 2 : 1))
    k_step_lanes(const Consts<T> g, const PPtrs<T> P, const FPtrs<T> F, const JPtrs<T> J, const SpeciesConst sc,
                 unsigned long long* counters, const WorkItem* items, const uint32_t* dense_idx,
                 const uint32_t* n_dense_ptr, const uint32_t* offsets, int nt2, int use_tma,
                 const __grid_constant__ FieldMaps maps) {
  constexpr int NT = kLThreads<T>;
  constexpr int PB = kLPB<T>;                          // particles per block: 4 (FP32) or 2 (FP64)
  extern __shared__ __align__(128) unsigned char smem_raw_[];
  T* sW = reinterpret_cast<T*>(smem_raw_);            // raw stencil first, then the lane windows [slot][thread]
  T* sN = sW + kLVals * NT;                           // node-major averaged fields
  T* sR = sN + kNodeElems<T>;                            // staged real columns [7][thread][PB]: dx1 dx2 u1 u2 u3 phi w
  int32_t* sI = reinterpret_cast<int32_t*>(sR + 7 * PB * NT);  // staged cell indices [2][thread][PB]
  uint64_t* bar = reinterpret_cast<uint64_t*>(sI + 2 * PB * NT);
  uint32_t* sO = reinterpret_cast<uint32_t*>(bar + 2);         // first slot of each of the tile's 256 sort keys, + end

  if (blockIdx.x >= n_dense_ptr[0]) return;
  const int tid = threadIdx.x;
  const WorkItem item = items[dense_idx[blockIdx.x]];
  const int c1lo = (int)(item.tile / (uint32_t)nt2) * kTile - kHalo;   // field window origin, cells
  const int c2lo = (int)(item.tile % (uint32_t)nt2) * kTile - kHalo;
  const int a2lo = c2lo - 1 + g.ng;
  const int off2 = ((a2lo % 4) + 4) % 4;

  for (int e = tid; e <= kTile * kTile; e += NT) sO[e] = __ldg(offsets + (size_t)item.tile * (kTile * kTile) + e);
  // ---- 1. stage the field stencil (as k_step_tiled) ----
  if (use_tma) {
    if (tid == 0) {
      mbar_init(bar, 1);
      mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
      mbar_expect_tx(bar, 6u * kWinF * kRowF * (uint32_t)sizeof(T));
#pragma unroll
      for (int c = 0; c < 6; ++c) tma_load_2d(sW + c * kRawComp, &maps.m[c], a2lo - off2, c1lo - 1 + g.ng, bar);
    }
    mbar_wait(bar, 0);
  } else {
    const int rows = g.n1 + 2 * g.ng;
    for (int e = tid; e < kRawElems; e += NT) {
      const int c = e / kRawComp, rem = e % kRawComp;
      const int a1 = c1lo - 1 + g.ng + rem / kRowF, a2 = a2lo - off2 + rem % kRowF;
      sW[e] = (a1 >= 0 && a1 < rows && a2 >= 0 && a2 < g.ld) ? __ldg(F.f[c] + (int64_t)a1 * g.ld + a2) : T(0);
    }
    __syncthreads();
  }
  // ---- 2. Yee samples -> nodes (R-S4), node-major ----
  for (int n = tid; n < kNodeW * kNodeW; n += NT) {
    const int w1 = n / kNodeW, w2 = n % kNodeW;
    const RawAcc<T> acc{sW, w1 + 1, w2 + 1 + off2};
    T* o = sN + n * kNodeStride<T>;
#pragma unroll
    for (int c = 0; c < 6; ++c) o[c] = node_value<T>(acc, c, yee_kind(c), 0, 0);
    if (kNodeStride<T> == 8) { o[6] = T(0); o[7] = T(0); }
  }
  __syncthreads();
  T* const pW = sW + tid;                              // this lane's window: slot s at pW[s * NT]
#pragma unroll 4
  for (int s = 0; s < kLVals; ++s) pW[s * NT] = T(0);

  // ---- 3. this lane's run: blocks of four particles, 16-byte aligned in every column ----
  const T eps = sc.massive ? T(1) : T(0);
  const T dt = (T)sc.dt;
  const T inv_dt = T(1) / dt;
  const T chg = (T)sc.charge;
  const uint32_t begin = item.begin, end = item.begin + item.count;
  const uint32_t B0 = begin / PB, B1 = (end + PB - 1u) / PB;
  const uint32_t bpl = (B1 - B0 + NT - 1) / NT;        // blocks per lane
  // kLQuad consecutive lanes share a contiguous region of kLQuad * bpl blocks and take its blocks in turn: one warp
  // instruction then reads (writes) kLQuad * 16 contiguous bytes per group - whole 32-byte sectors and whole
  // DRAM fetch units, used at once; a lane's own blocks stay within that one short region (about one sorted cell)
  const uint32_t b_first = B0 + (uint32_t)(tid / kLQuad) * (bpl * kLQuad) + (uint32_t)(tid % kLQuad);
  // processing order of the four staged particles: slot = j ^ swz makes the scalar staging reads of a warp
  // hit 32 different banks
  const int swz = (tid >> 3) & (PB - 1);
  T* const myR = sR + tid * PB;                        // column c at myR[c * PB * NT + slot]
  int32_t* const myI = sI + tid * PB;
  unsigned n_alive = 0, n_in = 0, n_out = 0, n_over = 0;
  // The window follows the SORTED cell of the run: the particles of one sort key are contiguous, and
  // offsets[key] (the scanned histogram of the sort, kept per species) is where each key starts, so the lane knows
  // the cell its current block was sorted into - with "sort_lookahead" the cell the particles are predicted to
  // pass in the middle of the sort interval, around which they are spread evenly before and after.
  bool have_win = false;
  int wo1 = 0, wo2 = 0;                                // window origin (cell): cells wo .. wo + 2, nodes wo .. wo + 3
  const uint32_t* const offs = sO;                     // keys of this tile: offs[0 .. 256]
  uint32_t key = 0, next_b = 0;
  if (b_first < B1) {                                  // key of the run's first particle: offs[key] <= k < offs[key + 1]
    const uint32_t kf = max(b_first * PB, begin);
    uint32_t lo = 0, hi = kTile * kTile;
#pragma unroll 1
    while (hi - lo > 1u) {
      const uint32_t mid = (lo + hi) >> 1;
      if (offs[mid] <= kf) lo = mid; else hi = mid;
    }
    key = lo;
    next_b = offs[key + 1];
  }
  const int t1c = (int)(item.tile / (uint32_t)nt2) * kTile, t2c = (int)(item.tile % (uint32_t)nt2) * kTile;
  const T* const rcol[7] = {P.dx1, P.dx2, P.u1, P.u2, P.u3, P.phi, P.w};
  T* const wcol[6] = {P.dx1, P.dx2, P.u1, P.u2, P.u3, P.phi};

  for (uint32_t b = b_first, bi = 0; bi < bpl && b < B1; ++bi, b += kLQuad) {
    const uint32_t k0 = b * PB;
    const bool full = k0 >= begin && k0 + PB <= end;
    {                                                  // move the window to the sorted cell of this block
      const uint32_t kb = max(k0, begin);
      while (kb >= next_b) { ++key; next_b = offs[key + 1]; }
      const int n1 = t1c + (int)(key >> 4) - 1, n2 = t2c + (int)(key & 15u) - 1;
      if (have_win && (n1 != wo1 || n2 != wo2)) {
        if (n1 == wo1 && n2 == wo2 + 1) lane_flush_col(g, J, pW, wo1, wo2);
        else lane_flush(g, J, pW, wo1, wo2);
      }
      have_win = true;
      wo1 = n1; wo2 = n2;
    }
    // ---- stage in ----
    uint32_t tags;                                     // one byte per particle of the block
    if (full) {
      if (PB == 4) { cp_async16(myI, P.i1 + k0); cp_async16(myI + PB * NT, P.i2 + k0); }
      else { cp_async8(myI, P.i1 + k0); cp_async8(myI + PB * NT, P.i2 + k0); }
#pragma unroll
      for (int c = 0; c < 7; ++c)
        if (c != 5 || sc.has_phi) cp_async16(myR + c * PB * NT, rcol[c] + k0);
      tags = PB == 4 ? *reinterpret_cast<const uint32_t*>(P.tag + k0) : (uint32_t)*reinterpret_cast<const uint16_t*>(P.tag + k0);
      if (kLPrefetch && (tid & 1) == 0 && bi + 1 < bpl && b + kLQuad < B1) {   // this lane's next block: in L2 by then
        constexpr uint32_t nx = PB * kLQuad;
        prefetch_l2(P.i1 + k0 + nx); prefetch_l2(P.i2 + k0 + nx);
#pragma unroll
        for (int c = 0; c < 7; ++c)
          if (c != 5 || sc.has_phi) prefetch_l2(rcol[c] + k0 + nx);
      }
      cp_async_wait_all();
    } else {
      tags = 0;
#pragma unroll
      for (int s = 0; s < PB; ++s) {
        const uint32_t k = k0 + s;
        if (k >= begin && k < end) {
          myI[s] = P.i1[k]; myI[PB * NT + s] = P.i2[k];
#pragma unroll
          for (int c = 0; c < 7; ++c)
            if (c != 5 || sc.has_phi) myR[c * PB * NT + s] = rcol[c][k];
          tags |= (uint32_t)P.tag[k] << (8 * s);
        }
      }
    }
    // ---- the particles of the block ----
#pragma unroll 1
    for (int j = 0; j < PB; ++j) {
      const int s = j ^ swz;
      if (((tags >> (8 * s)) & 0xffu) == 0u) continue;  // dead, or not of this item
      const uint32_t k = k0 + s;
      PState<T> p;
      p.i1 = myI[s]; p.i2 = myI[PB * NT + s];
      p.dx1 = myR[s]; p.dx2 = myR[PB * NT + s];
      p.u1 = myR[2 * PB * NT + s]; p.u2 = myR[3 * PB * NT + s]; p.u3 = myR[4 * PB * NT + s];
      const int ia = p.i1, ja = p.i2;
      const T xa = p.dx1, ya = p.dx2;
      if (P.i1p) { P.i1p[k] = ia; P.i2p[k] = ja; P.dx1p[k] = xa; P.dx2p[k] = ya; }
      const int wa1 = ia - c1lo, wa2 = ja - c2lo;      // cell inside the field window?
      const bool a_in = (unsigned)wa1 < (unsigned)kWinC && (unsigned)wa2 < (unsigned)kWinC;
      T Dp[3], Bp[3];
      if (a_in) {
        interp_nodes(sN, wa1 * kNodeW + wa2, p.dx1, p.dx2, Dp, Bp);
      } else {
        GlobalFieldAcc<T> acc{F, (int64_t)(ia + g.ng) * g.ld + (ja + g.ng), g.ld};
        interp_fields(acc, p.dx1, p.dx2, Dp, Bp);
      }
      T dphidt;
      bool reflected;
      const int res = push_particle<T, CoordT>(g, p, true, Dp, Bp, (T)sc.q_over_m, eps, dt, dphidt, reflected);
      n_alive += (res == 0); n_in += (res == 1); n_out += (res == 2);
      const int di = p.i1 - ia, dj = p.i2 - ja;
      const bool over = di > 1 || di < -1 || dj > 1 || dj < -1;
      const bool dep = res == 0 && !over;
      // the window slots of the start cell are requested now; the write-back of the particle and the arithmetic of
      // the deposit run while they arrive
      const bool a_win = dep && (unsigned)(ia - wo1) < (unsigned)kLWin && (unsigned)(ja - wo2) < (unsigned)kLWin;
      LaneCell<T> wa;
      if (a_win) wa.load(pW, ia, ja);
      myI[s] = p.i1; myI[PB * NT + s] = p.i2;
      myR[s] = p.dx1; myR[PB * NT + s] = p.dx2;
      myR[2 * PB * NT + s] = p.u1; myR[3 * PB * NT + s] = p.u2; myR[4 * PB * NT + s] = p.u3;
      if (sc.has_phi) myR[5 * PB * NT + s] += dt * dphidt;
      if (res != 0) { tags &= ~(0xffu << (8 * s)); continue; }
      if (over) { ++n_over; continue; }
      T v3 = dphidt;
      if (reflected)
        v3 = v3_at_path_midpoint<T, CoordT>(g, ia, ja, T(0.5) * (xa + (T)di + p.dx1), T(0.5) * (ya + (T)dj + p.dx2),
                                            p.u1, p.u2, p.u3, eps);
      const T qw = chg * myR[6 * PB * NT + s];
      T seg[2][8];
      deposit_segments(di, dj, xa, ya, p.dx1, p.dx2, qw * inv_dt, qw, v3, seg);
      const bool cross = (di != 0) || (dj != 0);
      if (!cross) {
#pragma unroll
        for (int q = 0; q < 8; ++q) seg[0][q] += seg[1][q];
      }
      // into the lane's window where the path lies inside it; a stray (drift since the sort) goes to L2 directly
      if (a_win)
        wa.add_store(seg[0]);
      else
        global_add8(J, (int64_t)(ia + g.ng) * g.ld + (ja + g.ng), g.ld, seg[0]);
      if (cross) {
        const int ib = ia + di, jb = ja + dj;
        if ((unsigned)(ib - wo1) < (unsigned)kLWin && (unsigned)(jb - wo2) < (unsigned)kLWin)
          lane_add8(pW, ib, jb, seg[1]);
        else
          global_add8(J, (int64_t)(ib + g.ng) * g.ld + (jb + g.ng), g.ld, seg[1]);
      }
    }
    // ---- stage out ----
    if (full) {
      if (PB == 4) {
        *reinterpret_cast<uint4*>(P.i1 + k0) = *reinterpret_cast<const uint4*>(myI);
        *reinterpret_cast<uint4*>(P.i2 + k0) = *reinterpret_cast<const uint4*>(myI + PB * NT);
        *reinterpret_cast<uint32_t*>(P.tag + k0) = tags;
      } else {
        *reinterpret_cast<uint2*>(P.i1 + k0) = *reinterpret_cast<const uint2*>(myI);
        *reinterpret_cast<uint2*>(P.i2 + k0) = *reinterpret_cast<const uint2*>(myI + PB * NT);
        *reinterpret_cast<uint16_t*>(P.tag + k0) = (uint16_t)tags;
      }
#pragma unroll
      for (int c = 0; c < 6; ++c)
        if (c != 5 || sc.has_phi)
          *reinterpret_cast<uint4*>(wcol[c] + k0) = *reinterpret_cast<const uint4*>(myR + c * PB * NT);
    } else {
#pragma unroll
      for (int s = 0; s < PB; ++s) {
        const uint32_t k = k0 + s;
        if (k >= begin && k < end) {
          P.i1[k] = myI[s]; P.i2[k] = myI[PB * NT + s];
#pragma unroll
          for (int c = 0; c < 6; ++c)
            if (c != 5 || sc.has_phi) wcol[c][k] = myR[c * PB * NT + s];
          P.tag[k] = (uint8_t)((tags >> (8 * s)) & 0xffu);
        }
      }
    }
  }
  if (have_win) lane_flush(g, J, pW, wo1, wo2);
  // counters: one atomic per warp and counter
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    n_alive += __shfl_xor_sync(0xffffffffu, n_alive, o);
    n_in += __shfl_xor_sync(0xffffffffu, n_in, o);
    n_out += __shfl_xor_sync(0xffffffffu, n_out, o);
    n_over += __shfl_xor_sync(0xffffffffu, n_over, o);
  }
  if ((tid & 31) == 0) {
    if (n_alive) atomicAdd(&counters[0], (unsigned long long)n_alive);
    if (n_in) atomicAdd(&counters[1], (unsigned long long)n_in);
    if (n_out) atomicAdd(&counters[2], (unsigned long long)n_out);
    if (n_over) atomicAdd(&counters[3], (unsigned long long)n_over);
    if (n_alive + n_in + n_out) atomicAdd(&counters[4], (unsigned long long)(n_alive + n_in + n_out));
  }
}

template <typename T, typename CoordT = Coord<T>>
bool launch_step_lanes(const TmaEncoder& enc, bool want_tma, const Consts<T>& g, const PPtrs<T>& P, const FPtrs<T>& F,
                       const JPtrs<T>& J, const SpeciesConst& sc, unsigned long long* counters, const WorkItem* items,
                       const uint32_t* dense_idx, const uint32_t* d_n_dense, const uint32_t* offsets, uint32_t max_dense,
                       bool& attr_set,
                       cudaStream_t st, std::string& err) {
  if (!attr_set) {
    cudaError_t ea = cudaFuncSetAttribute(k_step_lanes<T, CoordT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)lanes_smem_bytes<T>());
    if (ea != cudaSuccess) {
      err = std::string("k_step_lanes shared-memory opt-in: ") + cudaGetErrorString(ea);
      return false;
    }
    attr_set = true;
  }
  FieldMaps maps;
  memset(&maps, 0, sizeof(maps));
  int use_tma = want_tma ? 1 : 0;
  const int rows = g.n1 + 2 * g.ng;
  for (int c = 0; c < 6 && use_tma; ++c)
    if (!enc.encode(&maps.m[c], F.f[c], (int)sizeof(T), rows, g.ld)) use_tma = 0;
  const int nt2 = (g.n2 + kTile - 1) / kTile;
  k_step_lanes<T, CoordT><<<max_dense, kLThreads<T>, lanes_smem_bytes<T>(), st>>>(g, P, F, J, sc, counters, items, dense_idx,
                                                                              d_n_dense, offsets, nt2, use_tma, maps);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    err = std::string("k_step_lanes launch: ") + cudaGetErrorString(e);
    return false;
  }
  return true;
}

}  // namespace grpic
