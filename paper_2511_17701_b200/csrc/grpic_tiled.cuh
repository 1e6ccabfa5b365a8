// grpic_tiled.cuh — the fused step over cell-sorted tiles.
//
// One CTA per work item (tile, particle range <= kChunk) of the table grpic_sort built:
//   1. one elected thread issues six 2-D TMA loads (cp.async.bulk.tensor) that bring the tile's
//      field stencil — (kTile + 2 kHalo + 2) x (kTile + 2 kHalo + 6) samples of each of D1 D2 D3 B1 B2 B3 — into shared
//      memory, completion tracked by an mbarrier; out-of-range rows/columns are zero-filled by TMA;
//   2. every thread pushes its particles (steps 1-11 + BCs) with the gather served from shared
//      memory; a particle that has drifted out of the window since the last sort falls back to
//      global gathers, so the result never depends on how stale the table is;
//   3. J is accumulated in a shared-memory tile: contributions of lanes that deposit into the same
//      cell are first summed across the warp (segmented shuffle reduction over runs of equal cell),
//      then one lane per run issues the shared atomics; particles leaving the window use global
//      reductions;
//   4. one flush of the non-zero shared J entries to HBM with red.global.add.
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

// ---- shared-memory accessors ----
template <typename T>
struct SmemFieldAcc {
  const T* base;  // sample (c1, c2) of component 0, i.e. the particle's own cell
  __device__ __forceinline__ T operator()(int c, int di, int dj) const {
    return base[c * (kWinF * kRowF) + di * kRowF + dj];
  }
};

__device__ __forceinline__ void smem_add(float* p, float v) { atomicAdd(p, v); }
__device__ __forceinline__ void smem_add(double* p, double v) { atomicAdd(p, v); }

constexpr int kJStride = kWinF;                 // row stride of the shared J tile
constexpr int kJComp = kWinJ * kJStride;        // one component

template <typename T>
__device__ __forceinline__ void smem_add8(T* sJ, int node, const T v[8]) {
  smem_add(sJ + node, v[0]);
  smem_add(sJ + node + 1, v[1]);
  smem_add(sJ + kJComp + node, v[2]);
  smem_add(sJ + kJComp + node + kJStride, v[3]);
  smem_add(sJ + 2 * kJComp + node, v[4]);
  smem_add(sJ + 2 * kJComp + node + kJStride, v[5]);
  smem_add(sJ + 2 * kJComp + node + 1, v[6]);
  smem_add(sJ + 2 * kJComp + node + kJStride + 1, v[7]);
}

template <typename T>
__device__ __forceinline__ void global_add8(const JPtrs<T>& J, int64_t k, int ld, const T v[8]) {
  red_add(J.j[0] + k, v[0]);
  red_add(J.j[0] + k + 1, v[1]);
  red_add(J.j[1] + k, v[2]);
  red_add(J.j[1] + k + ld, v[3]);
  red_add(J.j[2] + k, v[4]);
  red_add(J.j[2] + k + ld, v[5]);
  red_add(J.j[2] + k + 1, v[6]);
  red_add(J.j[2] + k + ld + 1, v[7]);
}

// Warp-aggregated flush of the per-lane run accumulators into the shared J tile: lanes holding the same
// cell key in consecutive lanes form a run; the run is summed with log2(32) shuffle steps and its first
// lane issues the eight shared atomics.  (Shared FP atomics are compare-and-swap loops on sm_100a —
// ATOMS.CAST.SPIN — so fewer, conflict-free atomics is what matters.)
template <typename T>
__device__ __forceinline__ void warp_flush_runs(T* sJ, int lane, bool valid, int node, T acc[8]) {
  const int key = valid ? node : (0x40000000 + lane);                 // idle lanes: unique keys
  const int key_prev = __shfl_up_sync(0xffffffffu, key, 1);
  const bool head = (lane == 0) || (key != key_prev);
  const unsigned heads = __ballot_sync(0xffffffffu, head);
  const unsigned above = heads & ~((2u << lane) - 1u);                // run heads strictly above my lane
  const int run_last = above ? (__ffs(above) - 2) : 31;               // last lane of my run
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const bool take = (lane + d) <= run_last;
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      const T o = __shfl_down_sync(0xffffffffu, acc[q], d);
      if (take) acc[q] += o;
    }
  }
  if (head && valid) smem_add8(sJ, node, acc);
}

template <typename T>
__global__ void __launch_bounds__(kBlock, (sizeof(T) == 4 ? 3 : 1)) k_step_tiled(const Consts<T> g, const PPtrs<T> P, const FPtrs<T> F,
                                                       const JPtrs<T> J, const SpeciesConst sc,
                                                       unsigned long long* counters, const WorkItem* items,
                                                       const uint32_t* n_items_ptr, uint32_t max_items,
                                                       int64_t n_at_sort, int nt2, int use_tma,
                                                       const __grid_constant__ FieldMaps maps) {
  __shared__ __align__(128) T sF[6 * kWinF * kRowF];
  __shared__ __align__(16) T sJ[3 * kJComp];
  __shared__ __align__(8) uint64_t bar;

  const int tid = threadIdx.x, lane = tid & 31;
  // ---- tail blocks: particles appended after the last sort -> direct path ----
  if (blockIdx.x >= max_items) {
    const int64_t k = n_at_sort + (int64_t)(blockIdx.x - max_items) * kBlock + tid;
    particle_direct<T, true>(g, P, F, J, sc, counters, k);
    return;
  }
  if (blockIdx.x >= n_items_ptr[0]) return;
  const WorkItem item = items[blockIdx.x];
  const int c1lo = (int)(item.tile / (uint32_t)nt2) * kTile - kHalo;   // window origin, cells
  const int c2lo = (int)(item.tile % (uint32_t)nt2) * kTile - kHalo;
  // first fetched column (array index): the window's first sample, rounded down to a multiple of 4
  // elements so that its byte address is 16-byte aligned (a TMA requirement on the innermost coordinate)
  const int a2lo = c2lo - 1 + g.ng;
  const int off2 = ((a2lo % 4) + 4) % 4;

  // ---- 1. stage the field stencil ----
  if (use_tma) {
    if (tid == 0) {
      mbar_init(&bar, 1);
      mbar_fence_init();
    }
    __syncthreads();
    if (tid == 0) {
      mbar_expect_tx(&bar, 6u * kWinF * kRowF * (uint32_t)sizeof(T));
#pragma unroll
      for (int c = 0; c < 6; ++c)
        tma_load_2d(sF + c * kWinF * kRowF, &maps.m[c], a2lo - off2, c1lo - 1 + g.ng, &bar);
    }
  } else {
    const int rows = g.n1 + 2 * g.ng;
    for (int e = tid; e < 6 * kWinF * kRowF; e += kBlock) {
      const int c = e / (kWinF * kRowF), rem = e % (kWinF * kRowF);
      const int a1 = c1lo - 1 + g.ng + rem / kRowF, a2 = a2lo - off2 + rem % kRowF;
      sF[e] = (a1 >= 0 && a1 < rows && a2 >= 0 && a2 < g.ld) ? __ldg(F.f[c] + (int64_t)a1 * g.ld + a2) : T(0);
    }
  }
  for (int e = tid; e < 3 * kJComp; e += kBlock) sJ[e] = T(0);
  __syncthreads();
  if (use_tma) mbar_wait(&bar, 0);

  // ---- 2./3. particles ----
  const T eps = sc.massive ? T(1) : T(0);
  const T dt = (T)sc.dt;
  const T inv_dt = T(1) / dt;
  const uint32_t end = item.begin + item.count;
  unsigned n_alive = 0, n_in = 0, n_out = 0, n_over = 0;
  // Each warp owns a CONTIGUOUS slice of the item (sorted by cell): different warps then work on
  // different cells, and consecutive iterations of one lane stay in the same cell, so contributions
  // are first accumulated per lane in registers (acc) and flushed only when some lane changes cell.
  const uint32_t per_warp = ((item.count + kBlock - 1) / kBlock) * 32u;
  const uint32_t w_begin = item.begin + (uint32_t)(tid >> 5) * per_warp;
  const uint32_t w_end = min(end, w_begin + per_warp);
  bool acc_valid = false;
  int acc_node = 0;
  T acc[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) acc[q] = T(0);
  for (uint32_t base = w_begin; base < w_end; base += 32u) {
    const uint32_t k = base + lane;
    const bool alive = k < w_end && P.tag[k] != 0;
    int res = -1;
    bool dep_smem = false, dep_cross = false;
    int node_a = 0x7fffffff, node_b = 0;
    T va[8], vb[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) va[q] = vb[q] = T(0);
    if (alive) {
      PState<T> p;
      p.i1 = P.i1[k]; p.i2 = P.i2[k];
      p.dx1 = P.dx1[k]; p.dx2 = P.dx2[k];
      p.u1 = P.u1[k]; p.u2 = P.u2[k]; p.u3 = P.u3[k];
      const int ia = p.i1, ja = p.i2;
      const T xa = p.dx1, ya = p.dx2;
      P.i1p[k] = ia; P.i2p[k] = ja; P.dx1p[k] = xa; P.dx2p[k] = ya;
      const int wa1 = ia - c1lo, wa2 = ja - c2lo;                       // cell inside the window?
      const bool a_in = (unsigned)wa1 < (unsigned)kWinC && (unsigned)wa2 < (unsigned)kWinC;
      const int64_t cell = (int64_t)(ia + g.ng) * g.ld + (ja + g.ng);
      T Dp[3], Bp[3];
      if (a_in) {
        SmemFieldAcc<T> acc{sF + (wa1 + 1) * kRowF + (wa2 + 1 + off2)};
        interp_fields(acc, p.dx1, p.dx2, Dp, Bp);
      } else {
        GlobalFieldAcc<T> acc{F, cell, g.ld};
        interp_fields(acc, p.dx1, p.dx2, Dp, Bp);
      }
      T dphidt;
      bool reflected;
      res = push_particle(g, p, true, Dp, Bp, (T)sc.q_over_m, eps, dt, dphidt, reflected);
      P.i1[k] = p.i1; P.i2[k] = p.i2; P.dx1[k] = p.dx1; P.dx2[k] = p.dx2;
      P.u1[k] = p.u1; P.u2[k] = p.u2; P.u3[k] = p.u3;
      if (sc.has_phi) P.phi[k] += dt * dphidt;
      if (res != 0) P.tag[k] = 0;
      if (res == 0) {
        const int di = p.i1 - ia, dj = p.i2 - ja;
        if (di > 1 || di < -1 || dj > 1 || dj < -1) {
          ++n_over;
        } else {
          T v3 = dphidt;
          if (reflected)
            v3 = v3_at_path_midpoint(g, ia, ja, T(0.5) * (xa + (T)di + p.dx1), T(0.5) * (ya + (T)dj + p.dx2), p.u1,
                                     p.u2, p.u3, eps);
          const T qw = (T)sc.charge * P.w[k];
          T seg[2][8];
          deposit_segments(di, dj, xa, ya, p.dx1, p.dx2, qw * inv_dt, qw, v3,
                           [&seg](int s, T a0, T a1, T b0, T b1, T c00, T c10, T c01, T c11) {
                             seg[s][0] = a0; seg[s][1] = a1; seg[s][2] = b0; seg[s][3] = b1;
                             seg[s][4] = c00; seg[s][5] = c10; seg[s][6] = c01; seg[s][7] = c11;
                           });
          const int wb1 = wa1 + di, wb2 = wa2 + dj;
          const bool b_in = (unsigned)wb1 < (unsigned)kWinC && (unsigned)wb2 < (unsigned)kWinC;
          if (a_in && b_in) {
            dep_smem = true;
            node_a = wa1 * kJStride + wa2;
            if (di == 0 && dj == 0) {
#pragma unroll
              for (int q = 0; q < 8; ++q) va[q] = seg[0][q] + seg[1][q];
            } else {
              dep_cross = true;
              node_b = wb1 * kJStride + wb2;
#pragma unroll
              for (int q = 0; q < 8; ++q) { va[q] = seg[0][q]; vb[q] = seg[1][q]; }
            }
          } else {
            global_add8(J, cell, g.ld, seg[0]);
            global_add8(J, cell + (int64_t)di * g.ld + dj, g.ld, seg[1]);
          }
        }
      }
      n_alive += (res == 0); n_in += (res == 1); n_out += (res == 2);
    }
    // ---- run accumulation: flush (warp-aggregated) when any lane leaves its cell ----
    const bool must_flush = acc_valid && (!dep_smem || node_a != acc_node);
    if (__any_sync(0xffffffffu, must_flush)) {
      warp_flush_runs(sJ, lane, acc_valid, acc_node, acc);
      acc_valid = false;
#pragma unroll
      for (int q = 0; q < 8; ++q) acc[q] = T(0);
    }
    if (dep_smem) {
      acc_valid = true;
      acc_node = node_a;
#pragma unroll
      for (int q = 0; q < 8; ++q) acc[q] += va[q];
      if (dep_cross) smem_add8(sJ, node_b, vb);
    }
  }
  if (__any_sync(0xffffffffu, acc_valid)) warp_flush_runs(sJ, lane, acc_valid, acc_node, acc);
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
  // ---- 4. flush ----
  __syncthreads();
  const int rows = g.n1 + 2 * g.ng;
  for (int e = tid; e < 3 * kJComp; e += kBlock) {
    const T v = sJ[e];
    if (v != T(0)) {
      const int c = e / kJComp, rem = e % kJComp;
      const int a1 = c1lo + g.ng + rem / kJStride, a2 = c2lo + g.ng + rem % kJStride;
      if (a1 >= 0 && a1 < rows && a2 >= 0 && a2 < g.ld) red_add(J.j[c] + (int64_t)a1 * g.ld + a2, v);
    }
  }
}

template <typename T>
bool launch_step_tiled(const TmaEncoder& enc, bool want_tma, const Consts<T>& g, const PPtrs<T>& P, const FPtrs<T>& F,
                       const JPtrs<T>& J, const SpeciesConst& sc, unsigned long long* counters,
                       const WorkItem* items, const uint32_t* d_n_items, uint32_t max_items, int64_t n_at_sort,
                       cudaStream_t st, std::string& err) {
  FieldMaps maps;
  memset(&maps, 0, sizeof(maps));
  int use_tma = want_tma ? 1 : 0;
  const int rows = g.n1 + 2 * g.ng;
  for (int c = 0; c < 6 && use_tma; ++c)
    if (!enc.encode(&maps.m[c], F.f[c], (int)sizeof(T), rows, g.ld)) use_tma = 0;
  const int nt2 = (g.n2 + kTile - 1) / kTile;
  const int64_t tail = P.n > n_at_sort ? P.n - n_at_sort : 0;
  const unsigned grid = max_items + (unsigned)((tail + kBlock - 1) / kBlock);
  k_step_tiled<T><<<grid, kBlock, 0, st>>>(g, P, F, J, sc, counters, items, d_n_items, max_items, n_at_sort, nt2,
                                           use_tma, maps);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) {
    err = std::string("k_step_tiled launch: ") + cudaGetErrorString(e);
    return false;
  }
  return true;
}

}  // namespace grpic
