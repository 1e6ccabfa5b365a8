// grpic_tiled.cuh — the fused step over cell-sorted tiles.
//
// One CTA per work item (tile, particle range <= kChunk) of the table grpic_sort built:
//   1. one elected thread issues six 2-D TMA loads (cp.async.bulk.tensor) that bring the tile's
//      field stencil — (kTile + 2 kHalo + 2) x (kTile + 2 kHalo + 6) samples of each of D1 D2 D3 B1 B2 B3 — into shared
//      memory, completion tracked by an mbarrier; out-of-range rows/columns are zero-filled by TMA;
//   2. stage (i) of the gather (R-S4) is done ONCE per tile: the six Yee components are averaged to the
//      (kTile + 2 kHalo + 1)^2 nodes of the window and stored node-major (8 reals per node), so that a
//      particle's gather is four 32/64-byte node reads and six bilinear forms; the columns of the next 32
//      particles are requested before the current 32 are pushed (software pipeline);
//   3. every thread pushes its particles (steps 1-11 + BCs); a particle that has drifted out of the
//      window since the last sort falls back to global gathers, so the result never depends on how
//      stale the table is;
//   4. J is accumulated in shared memory, one PRIVATE tile per warp.  Shared FP atomics are
//      compare-and-swap loops on sm_100a (LDS + FADD + ATOMS.CAST.SPIN + BRA, retried on every address
//      collision); with a tile per warp none is needed: lanes depositing into the same cell are
//      summed across the warp first (transposing butterfly, 9 shuffles instead of 40, for groups of
//      kBigGroup or more lanes); stragglers (smaller groups, the part of a path in a neighbour cell) wait
//      in a per-warp queue and are resolved 32 at a time (butterfly again where they share a cell,
//      rank-by-rank rounds otherwise); what is left are plain read-modify-writes whose lanes never
//      share an address.  Particles leaving the window use global reductions;
//   5. one flush: the private tiles are summed and the non-zero entries go to HBM with red.global.add.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

#include "grpic_kernels.cuh"

namespace grpic {

// ---- TMA descriptor encoding through the driver entry point (no link-time libcuda dependency) ----
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

struct TmaEncoder {
  PFN_encodeTiled fn = nullptr;
  void init() {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (PFN_encodeTiled)p;
    else
      cudaGetLastError();
  }
  // [rows][ld] array of `elem_bytes`-wide floats, box kWinF rows x kRowF columns
  bool encode(CUtensorMap* m, const void* base, int elem_bytes, int rows, int ld) const {
    if (!fn) return false;
    if (((uintptr_t)base & 15u) || (((size_t)ld * elem_bytes) & 15u)) return false;
    cuuint64_t dims[2] = {(cuuint64_t)ld, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)ld * elem_bytes};
    cuuint32_t box[2] = {(cuuint32_t)kRowF, (cuuint32_t)kWinF};
    cuuint32_t estr[2] = {1, 1};
    return fn(m, elem_bytes == 4 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2,
              const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
  }
};

struct alignas(64) FieldMaps {
  CUtensorMap m[6];
};

// ---- mbarrier / TMA PTX ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::"r"(
          smem_u32(smem_dst)),
      "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1)
      : "memory");
}

// ---- launch shape of the tiled kernel ----
#ifndef GRPIC_TILED_BLOCK
#define GRPIC_TILED_BLOCK 128   // threads per CTA
#endif
#ifndef GRPIC_TILED_MINB
#define GRPIC_TILED_MINB 4      // resident CTAs per SM the FP32 kernel is compiled for (128 registers: no spills, room for the prefetch)
#endif
constexpr int kTBlock = GRPIC_TILED_BLOCK;

// ---- shared-memory layout ----
constexpr int kNodeW = kWinC + 1;               // nodes per window edge: c .. c+1                  (23)
// reals per node: D1 D2 D3 B1 B2 B3; FP32 pads to 8 (two 128-bit reads), FP64 keeps 6 (three 128-bit reads, 48 bytes)
#ifndef GRPIC_NODE_STRIDE32
#define GRPIC_NODE_STRIDE32 6
#endif
template <typename T> constexpr int kNodeStride = sizeof(T) == 4 ? GRPIC_NODE_STRIDE32 : 6;
constexpr int kJStride = (kWinJ + 3) / 4 * 4;   // row stride of one shared J tile                  (24)
constexpr int kJComp = kWinJ * kJStride;        // one component
constexpr int kJTile = 3 * kJComp;              // one private J tile (J1 J2 J3)
constexpr int kWarps = kTBlock / 32;
constexpr int kRawComp = (kWinF * kRowF + 31) / 32 * 32;   // one staged component; TMA wants 128-byte aligned destinations
constexpr int kRawElems = 6 * kRawComp;    // staged raw stencil; its space is reused by the J tiles after stage (i)
constexpr int kJElems = kWarps * kJTile;        // one PRIVATE J tile per warp: no atomics inside the CTA
constexpr int kFrontElems = kJElems > kRawElems ? kJElems : kRawElems;
template <typename T> constexpr int kNodeElems = (kNodeW * kNodeW * kNodeStride<T> + 3) / 4 * 4;   // what follows stays 16-byte aligned
static_assert(kJTile % 4 == 0 && kFrontElems % 4 == 0, "128-bit zero fill");

constexpr int kQueueVals = 8 * 64;            // reals per warp queue (8 x kQueue)
template <typename T>
constexpr size_t tiled_smem_bytes() {
  return (size_t)(kFrontElems + kNodeElems<T> + kWarps * kQueueVals) * sizeof(T) + (size_t)kWarps * 64 * sizeof(int) + 16;
}

// offset inside a shared J tile of value q (0..7, layout of deposit_segments) relative to the cell's node
__device__ __forceinline__ int j_offset_of(int q) {
  const int comp = (q < 2) ? 0 : ((q < 4) ? 1 : 2);
  const int d1 = (q == 3 || q == 5 || q == 7) ? kJStride : 0;
  const int d2 = (q == 1 || q == 6 || q == 7) ? 1 : 0;
  return comp * kJComp + d1 + d2;
}

template <typename T>
__device__ __forceinline__ T shfl_xor_(T v, int m) { return __shfl_xor_sync(0xffffffffu, v, m); }

// Eight plain read-modify-writes of one deposit segment into the warp's PRIVATE J tile, for all lanes
// with `on` at once.  Precondition: the lanes with `on` hold pairwise different cells (`node`).  Then the
// lanes of one instruction never share an address; addresses shared between DIFFERENT values of
// neighbouring cells (J1(c,c2+1) of cell c2 = J1(c,c2) of cell c2+1, ...) are kept apart by the four
// phases, each closed by __syncwarp() (memory ordering among the lanes of the warp).
template <typename T>
__device__ __forceinline__ void private_add8(T* sJ, bool on, int node, const T v[8]) {
  if (on) {
    sJ[node] += v[0];
    sJ[kJComp + node] += v[2];
    sJ[2 * kJComp + node] += v[4];
  }
  __syncwarp();
  if (on) {
    sJ[node + 1] += v[1];
    sJ[kJComp + node + kJStride] += v[3];
    sJ[2 * kJComp + node + kJStride] += v[5];
  }
  __syncwarp();
  if (on) sJ[2 * kJComp + node + 1] += v[6];
  __syncwarp();
  if (on) sJ[2 * kJComp + node + kJStride + 1] += v[7];
  __syncwarp();
}

// Warp-aggregated addition into the warp's private J tile.  Lanes with `has` hold a cell `key` (node index
// in the tile) and eight values.  __match_any_sync groups the lanes by cell.
//   - A group of kBigGroup or more lanes (cell-sorted particles: usually the whole warp) is summed by a
//     transposing butterfly: after the xor-16 step a lane keeps four of the eight partial sums, after
//     xor-8 two, after xor-4 one, then two plain steps — 9 shuffles, and the sum of value
//     q = 4*bit4 + 2*bit3 + bit2 ends in the lanes with those bits; the eight lanes with (lane & 3) == 0
//     add them to eight different addresses with ONE plain read-modify-write.
//   - The lanes of smaller groups are served by rank inside their group: round r takes the r-th lane of
//     every group, so the lanes of one round hold pairwise different cells (private_add8).
#ifndef GRPIC_BIG_GROUP
#define GRPIC_BIG_GROUP 6
#endif
constexpr int kBigGroup = GRPIC_BIG_GROUP;

// kRounds = false: only the big groups are added; the function returns true in the lanes it did not serve.
template <typename T, bool kRounds>
__device__ __forceinline__ bool warp_deposit(T* sJ, int lane, int my_off, bool has, int key, const T v[8]) {
  const unsigned act = __ballot_sync(0xffffffffu, has);
  if (act == 0u) return false;
  const unsigned peers = __match_any_sync(0xffffffffu, has ? key : ~lane);
  const int cnt = __popc(peers);
  unsigned big = __ballot_sync(0xffffffffu, has && cnt >= kBigGroup);
  const bool b4 = lane & 16, b3 = lane & 8, b2 = lane & 4;
  while (big) {
    const int leader = __ffs(big) - 1;
    const unsigned pm = __shfl_sync(0xffffffffu, peers, leader);
    const int k0 = __shfl_sync(0xffffffffu, key, leader);
    big &= ~pm;
    T x[4], y[2], z;
    if (pm == 0xffffffffu) {                       // the whole warp deposits into one cell: no masking
#pragma unroll
      for (int j = 0; j < 4; ++j) x[j] = (b4 ? v[j + 4] : v[j]) + shfl_xor_(b4 ? v[j] : v[j + 4], 16);
    } else {
      const bool mine = (pm >> lane) & 1u;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const T lo = mine ? v[j] : T(0), hi = mine ? v[j + 4] : T(0);
        x[j] = (b4 ? hi : lo) + shfl_xor_(b4 ? lo : hi, 16);
      }
    }
#pragma unroll
    for (int j = 0; j < 2; ++j) y[j] = (b3 ? x[j + 2] : x[j]) + shfl_xor_(b3 ? x[j] : x[j + 2], 8);
    z = (b2 ? y[1] : y[0]) + shfl_xor_(b2 ? y[0] : y[1], 4);
    z += shfl_xor_(z, 2);
    z += shfl_xor_(z, 1);
    if ((lane & 3) == 0) sJ[k0 + my_off] += z;
    __syncwarp();
  }
  const bool small = has && cnt < kBigGroup;
  if (!kRounds) return small;
  unsigned rem = __ballot_sync(0xffffffffu, small);
  if (rem) {
    const int rank = __popc(peers & ((1u << lane) - 1u));
    for (int r = 0; r < kBigGroup - 1 && rem; ++r) {
      const bool on = small && rank == r;
      private_add8(sJ, on, key, v);
      rem &= ~__ballot_sync(0xffffffffu, on);
    }
  }
  return false;
}

// Deferred stragglers.  Lanes whose cell is shared by fewer than kBigGroup lanes of the current 32 particles
// (particles that drifted out of their sorted cell, sparse cells) and the part of a path that lies in a
// neighbour cell are a few entries per iteration; resolving their conflicts every iteration costs as much
// as the whole push of a particle.  They are appended to a per-warp queue in shared memory (cell + eight
// values, structure of arrays) and resolved 32 at a time with one warp_deposit — where entries of the
// same cell collected over several iterations form big groups again.
constexpr int kQueue = 64;                      // entries per warp: at most 31 left over + 32 appended

template <typename T>
struct WarpQueue {
  int* k;      // [kQueue]
  T* v;        // [8][kQueue]
  int n;       // warp-uniform
  __device__ __forceinline__ void append(int lane, bool has, int key, const T val[8]) {
    const unsigned m = __ballot_sync(0xffffffffu, has);
    if (m == 0u) return;
    if (has) {
      const int pos = n + __popc(m & ((1u << lane) - 1u));
      k[pos] = key;
#pragma unroll
      for (int q = 0; q < 8; ++q) v[q * kQueue + pos] = val[q];
    }
    n += __popc(m);
    __syncwarp();
  }
  // resolve 32 entries from the top while at least `keep`+1 .. are queued: drain(31) keeps < 32, drain(0) empties
  __device__ __forceinline__ void drain(T* sJ, int lane, int my_off, int keep) {
    while (n > keep) {
      const int base = n > 32 ? n - 32 : 0;
      const bool has = base + lane < n;
      int key = 0;
      T val[8];
      if (has) {
        key = k[base + lane];
#pragma unroll
        for (int q = 0; q < 8; ++q) val[q] = v[q * kQueue + base + lane];
      }
      warp_deposit<T, true>(sJ, lane, my_off, has, key, val);
      n = base;
      __syncwarp();
    }
  }
};

// node-major shared field accessor: four node reads, six bilinear forms
template <typename T>
__device__ __forceinline__ void interp_nodes(const T* nod, int n00, T dx1, T dx2, T D[3], T B[3]) {
  T c[4][6];
  const int idx[4] = {n00, n00 + kNodeW, n00 + 1, n00 + kNodeW + 1};   // (0,0) (1,0) (0,1) (1,1)
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (sizeof(T) == 4 && kNodeStride<T> == 8) {
      const float4* p = reinterpret_cast<const float4*>(nod + idx[k] * kNodeStride<T>);
      const float4 a = p[0], b = p[1];
      c[k][0] = (T)a.x; c[k][1] = (T)a.y; c[k][2] = (T)a.z; c[k][3] = (T)a.w; c[k][4] = (T)b.x; c[k][5] = (T)b.y;
    } else if (sizeof(T) == 4) {
      const float2* p = reinterpret_cast<const float2*>(nod + idx[k] * kNodeStride<T>);
      const float2 a = p[0], b = p[1], d = p[2];
      c[k][0] = (T)a.x; c[k][1] = (T)a.y; c[k][2] = (T)b.x; c[k][3] = (T)b.y; c[k][4] = (T)d.x; c[k][5] = (T)d.y;
    } else {
      const double2* p = reinterpret_cast<const double2*>(nod + idx[k] * kNodeStride<T>);
      const double2 a = p[0], b = p[1], d = p[2];
      c[k][0] = (T)a.x; c[k][1] = (T)a.y; c[k][2] = (T)b.x; c[k][3] = (T)b.y; c[k][4] = (T)d.x; c[k][5] = (T)d.y;
    }
  }
  D[0] = bilinear(c[0][0], c[1][0], c[2][0], c[3][0], dx1, dx2);
  D[1] = bilinear(c[0][1], c[1][1], c[2][1], c[3][1], dx1, dx2);
  D[2] = bilinear(c[0][2], c[1][2], c[2][2], c[3][2], dx1, dx2);
  B[0] = bilinear(c[0][3], c[1][3], c[2][3], c[3][3], dx1, dx2);
  B[1] = bilinear(c[0][4], c[1][4], c[2][4], c[3][4], dx1, dx2);
  B[2] = bilinear(c[0][5], c[1][5], c[2][5], c[3][5], dx1, dx2);
}

template <typename T>
struct RawAcc {      // raw staged stencil: sample (row, col) of component c
  const T* raw;
  int row, col;
  __device__ __forceinline__ T operator()(int c, int di, int dj) const {
    return raw[c * kRawComp + (row + di) * kRowF + (col + dj)];
  }
};

// kDeposit = false is grpic_interp_push over the sorted tiles: the same kernel without steps 4-5.
template <typename T, typename CoordT = Coord<T>, bool kDeposit = true>
__global__ void __launch_bounds__(kTBlock, (sizeof(T) == 4 ? GRPIC_TILED_MINB : 1))
    k_step_tiled(const Consts<T> g, const PPtrs<T> P, const FPtrs<T> F, const JPtrs<T> J, const SpeciesConst sc,
                 unsigned long long* counters, const WorkItem* items, const uint32_t* n_items_ptr,
                 int nt2, int use_tma, int skip_dense,
                 const __grid_constant__ FieldMaps maps) {
  extern __shared__ __align__(128) unsigned char smem_raw_[];
  T* sF = reinterpret_cast<T*>(smem_raw_);            // raw stencil, later the kWarps private J tiles
  T* sN = sF + kFrontElems;                           // node-major averaged fields
  T* sQv = sN + kNodeElems<T>;                           // per-warp straggler queues: values, then cells
  int* sQk = reinterpret_cast<int*>(sQv + kWarps * kQueueVals);
  uint64_t* bar = reinterpret_cast<uint64_t*>(sQk + kWarps * kQueue);

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  T* sJ = sF + wid * kJTile;                          // this warp's private J tile
  // (slots behind the alive particles of the last sort: k_push_or_step_from, launched beside this kernel)
  if (blockIdx.x >= n_items_ptr[0]) return;
  const WorkItem item = items[blockIdx.x];
  if (skip_dense && item.pad) return;                 // a dense item: k_step_lanes has it (grpic_lanes.cuh)
  const int c1lo = (int)(item.tile / (uint32_t)nt2) * kTile - kHalo;   // window origin, cells
  const int c2lo = (int)(item.tile % (uint32_t)nt2) * kTile - kHalo;
  // first fetched column (array index): the window's first sample, rounded down to a multiple of 4
  // elements so that its byte address is 16-byte aligned (a TMA requirement on the innermost coordinate)
  const int a2lo = c2lo - 1 + g.ng;
  const int off2 = ((a2lo % 4) + 4) % 4;

  // ---- 1. stage the field stencil ----
  if (use_tma) {
    if (tid == 0) {
      mbar_init(bar, 1);
      mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
      mbar_expect_tx(bar, 6u * kWinF * kRowF * (uint32_t)sizeof(T));
#pragma unroll
      for (int c = 0; c < 6; ++c)
        tma_load_2d(sF + c * kRawComp, &maps.m[c], a2lo - off2, c1lo - 1 + g.ng, bar);
    }
    mbar_wait(bar, 0);
  } else {
    const int rows = g.n1 + 2 * g.ng;
    for (int e = tid; e < kRawElems; e += kTBlock) {
      const int c = e / kRawComp, rem = e % kRawComp;
      const int a1 = c1lo - 1 + g.ng + rem / kRowF, a2 = a2lo - off2 + rem % kRowF;
      sF[e] = (a1 >= 0 && a1 < rows && a2 >= 0 && a2 < g.ld) ? __ldg(F.f[c] + (int64_t)a1 * g.ld + a2) : T(0);
    }
    __syncthreads();
  }
  // ---- 2. stage (i) of the gather: Yee samples -> nodes (R-S4), node-major ----
  for (int n = tid; n < kNodeW * kNodeW; n += kTBlock) {
    const int w1 = n / kNodeW, w2 = n % kNodeW;
    const RawAcc<T> acc{sF, w1 + 1, w2 + 1 + off2};
    T* o = sN + n * kNodeStride<T>;
#pragma unroll
    for (int c = 0; c < 6; ++c) o[c] = node_value<T>(acc, c, yee_kind(c), 0, 0);
    if (kNodeStride<T> == 8) { o[6] = T(0); o[7] = T(0); }
  }
  __syncthreads();
  {                                                    // the raw stencil is dead: its space becomes the J tiles
    float4* z4 = reinterpret_cast<float4*>(sF);
    constexpr int n4 = (int)(kJElems * sizeof(T) / 16);
    for (int e = tid; e < n4; e += kTBlock) z4[e] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();

  // ---- 3./4. particles ----
  const T eps = sc.massive ? T(1) : T(0);
  const T dt = (T)sc.dt;
  const T inv_dt = T(1) / dt;
  const T chg = (T)sc.charge;
  const int my_off = j_offset_of(((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1));
  const uint32_t end = item.begin + item.count;
  unsigned n_alive = 0, n_in = 0, n_out = 0, n_over = 0;
  WarpQueue<T> Q{sQk + wid * kQueue, sQv + wid * kQueueVals, 0};
  // Each warp owns a CONTIGUOUS slice of the item (sorted by cell): the 32 particles of one iteration
  // then sit in one to three cells, which is what makes the warp-level aggregation cheap.
  const uint32_t per_warp = ((item.count + kTBlock - 1) / kTBlock) * 32u;
  const uint32_t w_begin = item.begin + (uint32_t)wid * per_warp;
  const uint32_t w_end = min(end, w_begin + per_warp);
  // Software pipeline: the columns of the NEXT 32 particles are requested before the current 32 are
  // pushed, so that their HBM latency is covered by ~1500 instructions of arithmetic.
  struct Cols {
    PState<T> p;
    T w, phi;
    uint8_t tg;
  };
  auto fetch = [&](uint32_t kk, bool ok, Cols& c) {
    c.tg = 0; c.w = T(0); c.phi = T(0);
    c.p.i1 = 0; c.p.i2 = 0; c.p.dx1 = c.p.dx2 = c.p.u1 = c.p.u2 = c.p.u3 = T(0);
    if (ok) {
      c.tg = P.tag[kk];
      c.p.i1 = P.i1[kk]; c.p.i2 = P.i2[kk];
      c.p.dx1 = P.dx1[kk]; c.p.dx2 = P.dx2[kk];
      c.p.u1 = P.u1[kk]; c.p.u2 = P.u2[kk]; c.p.u3 = P.u3[kk];
      c.w = P.w[kk];
      if (sc.has_phi) c.phi = P.phi[kk];
    }
  };
  Cols nxt;
  fetch(w_begin + lane, w_begin + lane < w_end, nxt);
  for (uint32_t base = w_begin; base < w_end; base += 32u) {
    const uint32_t k = base + lane;
    const bool in = k < w_end;
    PState<T> p = nxt.p;
    const T w = nxt.w, phi = nxt.phi;
    const uint8_t tg = nxt.tg;
    fetch(k + 32u, k + 32u < w_end, nxt);
    const bool alive = in && tg != 0;
    bool dep_a = false, dep_b = false;
    int node_a = 0, node_b = 0;
    T seg[2][8];
    if (alive) {
      const int ia = p.i1, ja = p.i2;
      const T xa = p.dx1, ya = p.dx2;
      if (!kDeposit || P.i1p) { P.i1p[k] = ia; P.i2p[k] = ja; P.dx1p[k] = xa; P.dx2p[k] = ya; }
      const int wa1 = ia - c1lo, wa2 = ja - c2lo;                       // cell inside the window?
      const bool a_in = (unsigned)wa1 < (unsigned)kWinC && (unsigned)wa2 < (unsigned)kWinC;
      const int64_t cell = (int64_t)(ia + g.ng) * g.ld + (ja + g.ng);
      T Dp[3], Bp[3];
      if (a_in) {
        interp_nodes(sN, wa1 * kNodeW + wa2, p.dx1, p.dx2, Dp, Bp);
      } else {
        GlobalFieldAcc<T> acc{F, cell, g.ld};
        interp_fields(acc, p.dx1, p.dx2, Dp, Bp);
      }
      T dphidt;
      bool reflected;
      const int res = push_particle<T, CoordT>(g, p, true, Dp, Bp, (T)sc.q_over_m, eps, dt, dphidt, reflected);
      P.i1[k] = p.i1; P.i2[k] = p.i2; P.dx1[k] = p.dx1; P.dx2[k] = p.dx2;
      P.u1[k] = p.u1; P.u2[k] = p.u2; P.u3[k] = p.u3;
      if (sc.has_phi) P.phi[k] = phi + dt * dphidt;
      if (res != 0) P.tag[k] = 0;
      if (kDeposit && res == 0) {
        const int di = p.i1 - ia, dj = p.i2 - ja;
        if (di > 1 || di < -1 || dj > 1 || dj < -1) {
          ++n_over;
        } else {
          T v3 = dphidt;
          if (reflected)
            v3 = v3_at_path_midpoint<T, CoordT>(g, ia, ja, T(0.5) * (xa + (T)di + p.dx1),
                                                T(0.5) * (ya + (T)dj + p.dx2), p.u1, p.u2, p.u3, eps);
          const T qw = chg * w;
          deposit_segments(di, dj, xa, ya, p.dx1, p.dx2, qw * inv_dt, qw, v3, seg);
          const int wb1 = wa1 + di, wb2 = wa2 + dj;
          const bool b_in = (unsigned)wb1 < (unsigned)kWinC && (unsigned)wb2 < (unsigned)kWinC;
          const bool cross = (di != 0) || (dj != 0);
          if (!cross) {
#pragma unroll
            for (int q = 0; q < 8; ++q) seg[0][q] += seg[1][q];
          }
          if (a_in && b_in) {
            dep_a = true;
            dep_b = cross;
            node_a = wa1 * kJStride + wa2;
            node_b = wb1 * kJStride + wb2;
          } else {
            global_add8(J, cell, g.ld, seg[0]);
            if (cross) global_add8(J, cell + (int64_t)di * g.ld + dj, g.ld, seg[1]);
          }
        }
      }
      n_alive += (res == 0); n_in += (res == 1); n_out += (res == 2);
    }
    if (kDeposit) {
      // big groups of the start cells now; stragglers and the neighbour-cell parts through the queue
      const bool left_a = warp_deposit<T, false>(sJ, lane, my_off, dep_a, node_a, seg[0]);
      Q.append(lane, left_a, node_a, seg[0]);
      Q.drain(sJ, lane, my_off, 31);
      Q.append(lane, dep_b, node_b, seg[1]);
      Q.drain(sJ, lane, my_off, 31);
    }
  }
  if (kDeposit) Q.drain(sJ, lane, my_off, 0);
  // counters: one atomic per warp and counter
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    n_alive += __shfl_xor_sync(0xffffffffu, n_alive, o);
    n_in += __shfl_xor_sync(0xffffffffu, n_in, o);
    n_out += __shfl_xor_sync(0xffffffffu, n_out, o);
    n_over += __shfl_xor_sync(0xffffffffu, n_over, o);
  }
  if (lane == 0) {
    if (n_alive) atomicAdd(&counters[0], (unsigned long long)n_alive);
    if (n_in) atomicAdd(&counters[1], (unsigned long long)n_in);
    if (n_out) atomicAdd(&counters[2], (unsigned long long)n_out);
    if (n_over) atomicAdd(&counters[3], (unsigned long long)n_over);
    if (n_alive + n_in + n_out) atomicAdd(&counters[4], (unsigned long long)(n_alive + n_in + n_out));
  }
  if (!kDeposit) return;
  // ---- 5. flush: sum the private tiles, one reduction per touched entry ----
  __syncthreads();
  const int rows = g.n1 + 2 * g.ng;
  for (int e = tid; e < kJTile; e += kTBlock) {
    T v = sF[e];
#pragma unroll
    for (int q = 1; q < kWarps; ++q) v += sF[q * kJTile + e];
    if (v != T(0)) {
      const int c = e / kJComp, rem = e % kJComp;
      const int a1 = c1lo + g.ng + rem / kJStride, a2 = c2lo + g.ng + rem % kJStride;
      if (a1 >= 0 && a1 < rows && a2 >= 0 && a2 < g.ld) red_add(J.j[c] + (int64_t)a1 * g.ld + a2, v);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// grpic_deposit over the sorted tiles: the deposit of (prev -> current) with the same per-warp private J tiles, warp
// aggregation and straggler queue as the fused step (steps 4-5 above); no field staging.  Items are the tiles of the
// last grpic_sort; the window test uses the PREVIOUS cell (the start of the path), like the fused kernel.
// The direct k_deposit sends every contribution to L2 with red.global.add: 13.5 ms for the 67 M particles of
// config 4 (hundreds of particles per cell hitting the same addresses); this kernel: see DESIGN.md section 7.
// ------------------------------------------------------------------------------------------------
template <typename T>
constexpr size_t deposit_smem_bytes() {
  return (size_t)(kJElems + kWarps * kQueueVals) * sizeof(T) + (size_t)kWarps * kQueue * sizeof(int);
}

template <typename T, typename CoordT = Coord<T>>
__global__ void __launch_bounds__(kTBlock, (sizeof(T) == 4 ? GRPIC_TILED_MINB : 2))
    k_deposit_tiled(const Consts<T> g, const PPtrs<T> P, const JPtrs<T> J, const SpeciesConst sc,
                    unsigned long long* counters, const WorkItem* items, const uint32_t* n_items_ptr, int nt2) {
  extern __shared__ __align__(128) unsigned char smem_raw_[];
  T* sF = reinterpret_cast<T*>(smem_raw_);
  T* sQv = sF + kJElems;
  int* sQk = reinterpret_cast<int*>(sQv + kWarps * kQueueVals);
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  T* sJ = sF + wid * kJTile;
  const T eps = sc.massive ? T(1) : T(0);
  const T inv_dt = T(1) / (T)sc.dt;
  const T chg = (T)sc.charge;
  unsigned n_over = 0;

  auto one = [&](int64_t k, bool in_window_ok, int c1lo, int c2lo, bool& dep_a, int& node_a, bool& dep_b, int& node_b,
                 T seg[2][8]) {
    dep_a = dep_b = false; node_a = node_b = 0;
    if (k >= P.n || P.tag[k] == 0) return;
    const int ia = P.i1p[k], ja = P.i2p[k];
    const int di = P.i1[k] - ia, dj = P.i2[k] - ja;
    if (di > 1 || di < -1 || dj > 1 || dj < -1) { ++n_over; return; }
    const T xa = P.dx1p[k], ya = P.dx2p[k], dx1 = P.dx1[k], dx2 = P.dx2[k];
    const T v3 = v3_at_path_midpoint<T, CoordT>(g, ia, ja, T(0.5) * (xa + (T)di + dx1), T(0.5) * (ya + (T)dj + dx2),
                                                P.u1[k], P.u2[k], P.u3[k], eps);
    const T qw = chg * P.w[k];
    deposit_segments(di, dj, xa, ya, dx1, dx2, qw * inv_dt, qw, v3, seg);
    const bool cross = (di != 0) || (dj != 0);
    if (!cross) {
#pragma unroll
      for (int q = 0; q < 8; ++q) seg[0][q] += seg[1][q];
    }
    const int64_t cell = (int64_t)(ia + g.ng) * g.ld + (ja + g.ng);
    const int wa1 = ia - c1lo, wa2 = ja - c2lo, wb1 = wa1 + di, wb2 = wa2 + dj;
    const bool a_in = in_window_ok && (unsigned)wa1 < (unsigned)kWinC && (unsigned)wa2 < (unsigned)kWinC;
    const bool b_in = in_window_ok && (unsigned)wb1 < (unsigned)kWinC && (unsigned)wb2 < (unsigned)kWinC;
    if (a_in && b_in) {
      dep_a = true; dep_b = cross;
      node_a = wa1 * kJStride + wa2; node_b = wb1 * kJStride + wb2;
    } else {
      global_add8(J, cell, g.ld, seg[0]);
      if (cross) global_add8(J, cell + (int64_t)di * g.ld + dj, g.ld, seg[1]);
    }
  };

  if (blockIdx.x >= n_items_ptr[0]) return;         // (slots the table does not cover: k_deposit_from)
  const WorkItem item = items[blockIdx.x];
  const int c1lo = (int)(item.tile / (uint32_t)nt2) * kTile - kHalo;
  const int c2lo = (int)(item.tile % (uint32_t)nt2) * kTile - kHalo;
  {
    float4* z4 = reinterpret_cast<float4*>(sF);
    constexpr int n4 = (int)(kJElems * sizeof(T) / 16);
    for (int e = tid; e < n4; e += kTBlock) z4[e] = make_float4(0.f, 0.f, 0.f, 0.f);
  }
  __syncthreads();
  const int my_off = j_offset_of(((lane >> 4) & 1) * 4 + ((lane >> 3) & 1) * 2 + ((lane >> 2) & 1));
  WarpQueue<T> Q{sQk + wid * kQueue, sQv + wid * kQueueVals, 0};
  const uint32_t end = item.begin + item.count;
  const uint32_t per_warp = ((item.count + kTBlock - 1) / kTBlock) * 32u;
  const uint32_t w_begin = item.begin + (uint32_t)wid * per_warp;
  const uint32_t w_end = min(end, w_begin + per_warp);
  for (uint32_t base = w_begin; base < w_end; base += 32u) {
    const uint32_t k = base + lane;
    bool dep_a, dep_b; int node_a, node_b; T seg[2][8];
    one(k < w_end ? (int64_t)k : (int64_t)P.n, true, c1lo, c2lo, dep_a, node_a, dep_b, node_b, seg);
    const bool left_a = warp_deposit<T, false>(sJ, lane, my_off, dep_a, node_a, seg[0]);
    Q.append(lane, left_a, node_a, seg[0]);
    Q.drain(sJ, lane, my_off, 31);
    Q.append(lane, dep_b, node_b, seg[1]);
    Q.drain(sJ, lane, my_off, 31);
  }
  Q.drain(sJ, lane, my_off, 0);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) n_over += __shfl_xor_sync(0xffffffffu, n_over, o);
  if (lane == 0 && n_over) atomicAdd(&counters[3], (unsigned long long)n_over);
  __syncthreads();
  const int rows = g.n1 + 2 * g.ng;
  for (int e = tid; e < kJTile; e += kTBlock) {
    T v = sF[e];
#pragma unroll
    for (int q = 1; q < kWarps; ++q) v += sF[q * kJTile + e];
    if (v != T(0)) {
      const int c = e / kJComp, rem = e % kJComp;
      const int a1 = c1lo + g.ng + rem / kJStride, a2 = c2lo + g.ng + rem % kJStride;
      if (a1 >= 0 && a1 < rows && a2 >= 0 && a2 < g.ld) red_add(J.j[c] + (int64_t)a1 * g.ld + a2, v);
    }
  }
}

template <typename T, typename CoordT = Coord<T>>
bool launch_deposit_tiled(const Consts<T>& g, const PPtrs<T>& P, const JPtrs<T>& J, const SpeciesConst& sc,
                          unsigned long long* counters, const WorkItem* items, const uint32_t* d_n_items,
                          uint32_t max_items, bool& attr_set, cudaStream_t st, std::string& err) {
  // attr_set: the shared-memory opt-in is per device and per loaded module; the flag lives in the context
  if (!attr_set) {
    cudaError_t ea = cudaFuncSetAttribute(k_deposit_tiled<T, CoordT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)deposit_smem_bytes<T>());
    if (ea != cudaSuccess) {
      err = std::string("k_deposit_tiled shared-memory opt-in: ") + cudaGetErrorString(ea);
      return false;
    }
    attr_set = true;
  }
  const int nt2 = (g.n2 + kTile - 1) / kTile;
  k_deposit_tiled<T, CoordT><<<max_items, kTBlock, deposit_smem_bytes<T>(), st>>>(g, P, J, sc, counters, items,
                                                                                 d_n_items, nt2);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    err = std::string("k_deposit_tiled launch: ") + cudaGetErrorString(e);
    return false;
  }
  return true;
}

template <typename T, typename CoordT = Coord<T>, bool kDeposit = true>
bool launch_step_tiled(const TmaEncoder& enc, bool want_tma, const Consts<T>& g, const PPtrs<T>& P, const FPtrs<T>& F,
                       const JPtrs<T>& J, const SpeciesConst& sc, unsigned long long* counters,
                       const WorkItem* items, const uint32_t* d_n_items, uint32_t max_items,
                       bool skip_dense, bool& attr_set, cudaStream_t st, std::string& err) {
  if (!attr_set) {
    cudaError_t ea = cudaFuncSetAttribute(k_step_tiled<T, CoordT, kDeposit>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                          (int)tiled_smem_bytes<T>());
    if (ea != cudaSuccess) {
      err = std::string("k_step_tiled shared-memory opt-in: ") + cudaGetErrorString(ea);
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
  k_step_tiled<T, CoordT, kDeposit><<<max_items, kTBlock, tiled_smem_bytes<T>(), st>>>(
      g, P, F, J, sc, counters, items, d_n_items, nt2, use_tma, skip_dense ? 1 : 0, maps);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    err = std::string("k_step_tiled launch: ") + cudaGetErrorString(e);
    return false;
  }
  return true;
}

}  // namespace grpic
