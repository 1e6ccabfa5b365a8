// grpic_kernels.cuh — the CUDA kernels behind include/grpic.h (sm_100a).
//
//   k_push_or_step<T,false,C>  steps 1-11 + particle BCs, one thread per particle    (grpic_interp_push, unsorted species)
//   k_push_or_step<T,true,C>   fused push + deposit, L2 gathers and red.global.add   (grpic_step, unsorted species;
//                              chunks of grpic_step_host; slots the tile table does not cover)
//   k_deposit<T,C>             charge-conserving deposit from (prev, current)        (grpic_deposit, unsorted species)
//   k_step_tiled<T,C,kDeposit> grpic_tiled.cuh: fused step over cell-sorted tiles — field stencil of the tile staged in
//                              shared memory by TMA, J in per-warp shared tiles, one flush (grpic_step; without the
//                              deposit half: grpic_interp_push on a sorted species)
//   k_deposit_tiled<T,C>       grpic_tiled.cuh: the deposit half alone               (grpic_deposit, sorted species)
//   k_step_lanes<T,C>          grpic_lanes.cuh: the fused step over the DENSE work items of a sorted species — one run of
//                              sorted particles per lane, lane-private J windows in shared memory, 128-bit column blocks
//                              (grpic_step; k_step_tiled keeps the sparse items)
//   k_push_or_step_from, k_deposit_from   the direct path over the slots behind the alive count of the last sort
//   k_probe<kind>              grpic_probe.cuh: throughput probes (measured roofline denominators)
//   k_sort_*, k_scan_*, k_items_*  counting sort by tile-major cell key + work-item table (grpic_sort)
//   grpic_fields.cuh           field-solver half: auxiliary fields, Faraday, Ampere, boundary conditions, filter
// C = coordinate class: Coord<T> (default map of the five configs, specialised) or CoordGen<T> (all maps of App. A).
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "grpic_device.cuh"

namespace grpic {

constexpr int kTile = 16;                       // cells per tile edge (sort key and shared-memory tile)
#ifndef GRPIC_HALO
#define GRPIC_HALO 3
#endif
constexpr int kHalo = GRPIC_HALO;               // extra cells around a tile served from shared memory
constexpr int kWinC = kTile + 2 * kHalo;        // cells per window edge                     (22)
constexpr int kWinF = kWinC + 2;                // field samples per window edge: c-1 .. c+1 (24)
constexpr int kRowF = (kWinF + 3 + 3) / 4 * 4;  // shared row length of the field window: TMA wants the first
                                                // column 16-byte aligned in global memory (up to 3 extra
                                                // columns on the left) and rows of whole 16 bytes       (28)
constexpr int kWinJ = kWinC + 1;                // J nodes per window edge: c .. c+1         (23)
#ifndef GRPIC_CHUNK
#define GRPIC_CHUNK 16384
#endif
constexpr int kChunk = GRPIC_CHUNK;             // max particles per work item
constexpr int kBlock = 256;

template <typename T>
struct PPtrs {
  int64_t n;
  int32_t *i1, *i2;
  T *dx1, *dx2, *u1, *u2, *u3, *phi;
  int32_t *i1p, *i2p;
  T *dx1p, *dx2p;
  const T* w;
  uint8_t* tag;
};
template <typename T>
struct FPtrs {
  const T* f[6];  // D1 D2 D3 B1 B2 B3
};
template <typename T>
struct JPtrs {
  T* j[3];
};
struct SpeciesConst {
  double q_over_m, charge, dt;
  int32_t massive, em, has_phi, do_deposit;
};

// counters: [0] alive after push, [1] absorbed inside, [2] absorbed outside, [3] overstep (most recent call);
// [4] particle updates since grpic_create (cumulative)
__device__ __forceinline__ void warp_count(unsigned long long* counters, int which, bool pred) {
  const unsigned m = __ballot_sync(0xffffffffu, pred);
  if (m && (threadIdx.x & 31) == 0) atomicAdd(&counters[which], (unsigned long long)__popc(m));
}

// global-memory field accessor
template <typename T>
struct GlobalFieldAcc {
  const FPtrs<T>& F;
  int64_t base;
  int ld;
  __device__ __forceinline__ T operator()(int c, int di, int dj) const {
    return __ldg(F.f[c] + base + (int64_t)di * ld + dj);
  }
};

// red.global.add: fire-and-forget reductions into the J arrays.  Written as PTX on an explicit global address:
// atomicAdd on a generic pointer makes ptxas emit, wherever it cannot prove the address space (the tiled kernels),
// a QSPC test plus a returning ATOM and two compare-and-swap loops per call site instead of one REDG.
__device__ __forceinline__ void red_add(float* p, float v) {
  asm volatile("red.global.add.f32 [%0], %1;" ::"l"(__cvta_generic_to_global(p)), "f"(v) : "memory");
}
__device__ __forceinline__ void red_add(double* p, double v) {
  asm volatile("red.global.add.f64 [%0], %1;" ::"l"(__cvta_generic_to_global(p)), "d"(v) : "memory");
}

// eight additions of one deposit segment (layout of deposit_segments' seg[s][0..7]) at cell offset k
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

// ------------------------------------------------------------------------------------------------
// shared per-particle driver used by k_push / k_step_direct
// ------------------------------------------------------------------------------------------------
template <typename T, bool kDeposit, typename CoordT = Coord<T>>
__device__ __forceinline__ void particle_direct(const Consts<T>& g, const PPtrs<T>& P, const FPtrs<T>& F,
                                                const JPtrs<T>& J, const SpeciesConst& sc,
                                                unsigned long long* counters, int64_t k) {
  const bool in_range = k < P.n;
  const bool alive = in_range && P.tag[k] != 0;
  int res = -1;
  bool over = false;
  if (alive) {
    PState<T> p;
    p.i1 = P.i1[k]; p.i2 = P.i2[k];
    p.dx1 = P.dx1[k]; p.dx2 = P.dx2[k];
    p.u1 = P.u1[k]; p.u2 = P.u2[k]; p.u3 = P.u3[k];
    const int ia = p.i1, ja = p.i2;
    const T xa = p.dx1, ya = p.dx2;
    // step 1
    if (!kDeposit || P.i1p) { P.i1p[k] = ia; P.i2p[k] = ja; P.dx1p[k] = xa; P.dx2p[k] = ya; }   // optional for the fused step
    T Dp[3] = {T(0), T(0), T(0)}, Bp[3] = {T(0), T(0), T(0)};
    const int64_t cell = (int64_t)(ia + g.ng) * g.ld + (ja + g.ng);
    if (sc.em) {
      GlobalFieldAcc<T> acc{F, cell, g.ld};
      interp_fields(acc, p.dx1, p.dx2, Dp, Bp);          // step 2
    }
    const T eps = sc.massive ? T(1) : T(0);
    const T dt = (T)sc.dt;
    T dphidt;
    bool reflected;
    res = push_particle<T, CoordT>(g, p, sc.em != 0, Dp, Bp, (T)sc.q_over_m, eps, dt, dphidt, reflected);
    P.i1[k] = p.i1; P.i2[k] = p.i2; P.dx1[k] = p.dx1; P.dx2[k] = p.dx2;
    P.u1[k] = p.u1; P.u2[k] = p.u2; P.u3[k] = p.u3;
    if (sc.has_phi) P.phi[k] += dt * dphidt;
    if (res != 0) P.tag[k] = 0;
    if (kDeposit && sc.do_deposit && res == 0) {
      const int di = p.i1 - ia, dj = p.i2 - ja;
      if (di > 1 || di < -1 || dj > 1 || dj < -1) {
        over = true;
      } else {
        T v3 = dphidt;
        if (reflected)
          v3 = v3_at_path_midpoint<T, CoordT>(g, ia, ja, T(0.5) * (xa + (T)di + p.dx1), T(0.5) * (ya + (T)dj + p.dx2),
                                              p.u1, p.u2, p.u3, eps);
        const T qw = (T)sc.charge * P.w[k];
        T seg[2][8];
        deposit_segments(di, dj, xa, ya, p.dx1, p.dx2, qw / dt, qw, v3, seg);
        if (di == 0 && dj == 0) {                          // both segments in one cell: one set of additions
#pragma unroll
          for (int q = 0; q < 8; ++q) seg[0][q] += seg[1][q];
          global_add8(J, cell, g.ld, seg[0]);
        } else {
          global_add8(J, cell, g.ld, seg[0]);
          global_add8(J, cell + (int64_t)di * g.ld + dj, g.ld, seg[1]);
        }
      }
    }
  }
  warp_count(counters, 0, res == 0);
  warp_count(counters, 1, res == 1);
  warp_count(counters, 2, res == 2);
  warp_count(counters, 4, res >= 0);
  if (kDeposit) warp_count(counters, 3, over);
}

template <typename T, bool kDeposit, typename CoordT = Coord<T>>
__global__ void __launch_bounds__(kBlock) k_push_or_step(const Consts<T> g, const PPtrs<T> P, const FPtrs<T> F,
                                                         const JPtrs<T> J, const SpeciesConst sc,
                                                         unsigned long long* counters) {
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  particle_direct<T, kDeposit, CoordT>(g, P, F, J, sc, counters, k);
}

// The same over the slots [*first_ptr, P.n) with *first_ptr read on the device: the slots behind the alive particles of
// the last sort (dead then, possibly revived or appended since), which the tile table does not cover.  Fixed grid,
// block-strided, so that the host never has to know the alive count (no read-back in grpic_sort).
template <typename T, bool kDeposit, typename CoordT = Coord<T>>
__global__ void __launch_bounds__(kBlock) k_push_or_step_from(const Consts<T> g, const PPtrs<T> P, const FPtrs<T> F,
                                                              const JPtrs<T> J, const SpeciesConst sc,
                                                              unsigned long long* counters, const uint32_t* first_ptr) {
  const int64_t first = (int64_t)first_ptr[0];
  for (int64_t base = first + (int64_t)blockIdx.x * kBlock; base < P.n; base += (int64_t)gridDim.x * kBlock)
    particle_direct<T, kDeposit, CoordT>(g, P, F, J, sc, counters, base + threadIdx.x);
}

// deposit from stored (prev, current) — Eq. 36 velocity recomputed at the path midpoint as the paper
// states it
template <typename T, typename CoordT = Coord<T>>
__device__ __forceinline__ void deposit_direct(const Consts<T>& g, const PPtrs<T>& P, const JPtrs<T>& J,
                                               const SpeciesConst& sc, unsigned long long* counters, int64_t k) {
  bool over = false;
  if (k < P.n && P.tag[k] != 0) {
    const int ia = P.i1p[k], ja = P.i2p[k];
    const int di = P.i1[k] - ia, dj = P.i2[k] - ja;
    if (di > 1 || di < -1 || dj > 1 || dj < -1) {
      over = true;
    } else {
      const T xa = P.dx1p[k], ya = P.dx2p[k], dx1 = P.dx1[k], dx2 = P.dx2[k];
      const T eps = sc.massive ? T(1) : T(0);
      const T v3 = v3_at_path_midpoint<T, CoordT>(g, ia, ja, T(0.5) * (xa + (T)di + dx1), T(0.5) * (ya + (T)dj + dx2), P.u1[k],
                                       P.u2[k], P.u3[k], eps);
      const T qw = (T)sc.charge * P.w[k];
      const int64_t cell = (int64_t)(ia + g.ng) * g.ld + (ja + g.ng);
      T seg[2][8];
      deposit_segments(di, dj, xa, ya, dx1, dx2, qw / (T)sc.dt, qw, v3, seg);
      global_add8(J, cell, g.ld, seg[0]);
      global_add8(J, cell + (int64_t)di * g.ld + dj, g.ld, seg[1]);
    }
  }
  warp_count(counters, 3, over);
}

template <typename T, typename CoordT = Coord<T>>
__global__ void __launch_bounds__(kBlock) k_deposit(const Consts<T> g, const PPtrs<T> P, const JPtrs<T> J,
                                                    const SpeciesConst sc, unsigned long long* counters) {
  deposit_direct<T, CoordT>(g, P, J, sc, counters, (int64_t)blockIdx.x * blockDim.x + threadIdx.x);
}
// slots [*first_ptr, P.n), see k_push_or_step_from
template <typename T, typename CoordT = Coord<T>>
__global__ void __launch_bounds__(kBlock) k_deposit_from(const Consts<T> g, const PPtrs<T> P, const JPtrs<T> J,
                                                         const SpeciesConst sc, unsigned long long* counters,
                                                         const uint32_t* first_ptr) {
  const int64_t first = (int64_t)first_ptr[0];
  for (int64_t base = first + (int64_t)blockIdx.x * kBlock; base < P.n; base += (int64_t)gridDim.x * kBlock)
    deposit_direct<T, CoordT>(g, P, J, sc, counters, base + threadIdx.x);
}

// ------------------------------------------------------------------------------------------------
// counting sort by tile-major cell key
// ------------------------------------------------------------------------------------------------
struct SortGeom {
  int32_t n1, n2, nt1, nt2;
  uint32_t n_keys;  // nt1*nt2*kTile*kTile + 1 (the last key is "dead")
};

__device__ __forceinline__ uint32_t tile_key(const SortGeom& s, int i1, int i2, bool alive) {
  if (!alive || i1 < 0 || i1 >= s.n1 || i2 < 0 || i2 >= s.n2) return s.n_keys - 1;
  const uint32_t t1 = (uint32_t)i1 / kTile, l1 = (uint32_t)i1 % kTile;
  const uint32_t t2 = (uint32_t)i2 / kTile, l2 = (uint32_t)i2 % kTile;
  return ((t1 * s.nt2 + t2) * kTile + l1) * kTile + l2;
}

// Look-ahead of the sort key ("sort_lookahead", include/grpic.h): the cell a particle is predicted to occupy after
// tau = L * dt of ballistic motion, dx^i/dt = alpha h^ij u_j / gamma - beta^i (Eq. 28) taken at its present place.
// This is an ORDERING HEURISTIC only - any order is a correct sort result, and the tile kernel treats a particle
// outside its tile's window through the global path - so it is written in plain FP32 with fast intrinsics in both
// builds and guards nothing but NaN.  With L = half the sort interval the particles of a warp are closest
// together in the middle of the interval instead of right after the sort, which halves the mean spread the
// warp-level deposit aggregation sees.
struct SortPredict {
  float tau, log_rmin, dxi, r_off, r_min, dr, deta, h0, a, mass, eps;
  int32_t r_lin, on;
};

__device__ __forceinline__ void predicted_cell(const SortPredict& q, int n1, int n2, int& i1, int& i2, float dx1,
                                               float dx2, float u1, float u2, float u3) {
  const float x1 = (float)i1 + dx1, x2 = (float)i2 + dx2;
  float r, s1;
  if (q.r_lin) {
    r = q.r_min + x1 * q.dr; s1 = q.dr;
  } else {
    const float rm = __expf(q.log_rmin + x1 * q.dxi);
    r = q.r_off + rm; s1 = q.dxi * rm;
  }
  const float pi = 3.14159265f;
  const float eta = x2 * q.deta, xx = eta * (1.0f / pi);
  const float th = eta + 2.0f * q.h0 * eta * (pi - 2.0f * eta) * (pi - eta) * (1.0f / (pi * pi));
  const float s2 = q.deta * (1.0f + 2.0f * q.h0 + 12.0f * q.h0 * xx * (xx - 1.0f));
  float sth, cth;
  __sincosf(th, &sth, &cth);
  const float s2th = fmaxf(sth * sth, 1e-8f);
  const float a2 = q.a * q.a, r2a2 = r * r + a2;
  const float Sigma = r * r + a2 * cth * cth, iSigma = __frcp_rn(Sigma), z = 2.0f * q.mass * r * iSigma;
  const float A = r2a2 * r2a2 - a2 * (r2a2 - 2.0f * q.mass * r) * s2th;
  const float h11 = s1 * s1 * (1.0f + z), h33 = A * s2th * iSigma, h13 = -s1 * q.a * (1.0f + z) * s2th;
  const float idet = __frcp_rn(h11 * h33 - h13 * h13);
  const float up1 = (h33 * u1 - h13 * u3) * idet, up3 = (h11 * u3 - h13 * u1) * idet, up2 = u2 * iSigma * __frcp_rn(s2 * s2);
  const float g2 = q.eps + up1 * u1 + up2 * u2 + up3 * u3;
  const float k = rsqrtf((1.0f + z) * fmaxf(g2, 1e-30f));           // alpha / gamma
  float p1 = x1 + q.tau * (k * up1 - __fdividef(z, (1.0f + z) * s1));
  float p2 = x2 + q.tau * (k * up2);
  if (p2 < 0.0f) p2 = -p2;
  if (p2 > (float)n2) p2 = 2.0f * (float)n2 - p2;
  if (p1 == p1 && p2 == p2) {
    i1 = min(max((int)floorf(p1), 0), n1 - 1);
    i2 = min(max((int)floorf(p2), 0), n2 - 1);
  }
}

#ifndef GRPIC_SORT_V
#define GRPIC_SORT_V 4
#endif
constexpr int kSortV = GRPIC_SORT_V;       // elements per thread of the histogram and rank kernels

// histogram: one atomic per run of equal keys inside a warp (sorted input -> few runs)
template <typename T>
__global__ void __launch_bounds__(kBlock) k_sort_hist(const SortGeom s, const SortPredict q, int64_t n, const int32_t* i1,
                                                      const int32_t* i2, const uint8_t* tag, const T* dx1, const T* dx2,
                                                      const T* u1, const T* u2, const T* u3, uint32_t* key_out,
                                                      uint32_t* hist) {
  // kSortV elements per thread, one block-wide stride apart: all loads are issued before the first vote
  const int64_t k0 = (int64_t)blockIdx.x * (kBlock * kSortV) + threadIdx.x;
  const int lane = threadIdx.x & 31;
  uint32_t key[kSortV];
#pragma unroll
  for (int v = 0; v < kSortV; ++v) {
    const int64_t k = k0 + v * kBlock;
    key[v] = 0xffffffffu;
    if (k < n) {
      int c1 = i1[k], c2 = i2[k];
      const bool alive = tag[k] != 0;
      if (q.on && alive && c1 >= 0 && c1 < s.n1 && c2 >= 0 && c2 < s.n2)
        predicted_cell(q, s.n1, s.n2, c1, c2, (float)dx1[k], (float)dx2[k], (float)u1[k], (float)u2[k], (float)u3[k]);
      key[v] = tile_key(s, c1, c2, alive);
    }
  }
#pragma unroll
  for (int v = 0; v < kSortV; ++v) {
    const int64_t k = k0 + v * kBlock;
    const bool in = k < n;
    if (in) key_out[k] = key[v];
    const unsigned peers = __match_any_sync(0xffffffffu, key[v]);
    if (in && lane == __ffs(peers) - 1) atomicAdd(&hist[key[v]], (uint32_t)__popc(peers));
  }
}

// rank of every particle inside its key: offset[key]++ (warp-aggregated); written as the inverse permutation
// src[slot] = particle, so that the move is a gather (coalesced writes, nearly sequential reads)
__global__ void __launch_bounds__(kBlock) k_sort_rank(int64_t n, const uint32_t* key_in, uint32_t* cursor,
                                                      uint32_t* dest) {
  const int64_t k0 = (int64_t)blockIdx.x * (kBlock * kSortV) + threadIdx.x;
  const int lane = threadIdx.x & 31;
  uint32_t key[kSortV], base[kSortV];
  unsigned peers[kSortV];
#pragma unroll
  for (int v = 0; v < kSortV; ++v) {
    const int64_t k = k0 + v * kBlock;
    key[v] = k < n ? key_in[k] : 0xffffffffu;
  }
#pragma unroll
  for (int v = 0; v < kSortV; ++v) {                       // the kSortV returning atomics are in flight together
    const bool in = k0 + v * kBlock < n;
    peers[v] = __match_any_sync(0xffffffffu, key[v]);
    base[v] = 0;
    if (in && lane == __ffs(peers[v]) - 1) base[v] = atomicAdd(&cursor[key[v]], (uint32_t)__popc(peers[v]));
  }
#pragma unroll
  for (int v = 0; v < kSortV; ++v) {
    const int64_t k = k0 + v * kBlock;
    const uint32_t b = __shfl_sync(0xffffffffu, base[v], __ffs(peers[v]) - 1);
    if (k < n) dest[b + __popc(peers[v] & ((1u << lane) - 1u))] = (uint32_t)k;   // dest[] holds the SOURCE of every slot
  }
}

// kGatherV destination slots per thread (one block-wide stride apart, so every access of a warp stays coalesced):
// the kGatherV source indices are loaded first and then kGatherV independent loads per column are in flight -
// the one-slot form left the memory system latency-bound at 43 % of the DRAM rate (ncu, config 4)
#ifndef GRPIC_GATHER_V
#define GRPIC_GATHER_V 4
#endif
constexpr int kGatherV = GRPIC_GATHER_V;

template <typename U>
__device__ __forceinline__ void gather_column(U* __restrict__ dst, const U* __restrict__ from,
                                              const uint32_t (&k)[kGatherV], const bool (&ok)[kGatherV], int64_t d0) {
  U r[kGatherV];
#pragma unroll
  for (int v = 0; v < kGatherV; ++v) r[v] = from[k[v]];
#pragma unroll
  for (int v = 0; v < kGatherV; ++v)
    if (ok[v]) dst[d0 + v * kBlock] = r[v];
}

template <typename T>
__global__ void __launch_bounds__(kBlock) k_sort_gather(const PPtrs<T> in, const PPtrs<T> out,
                                                        const uint32_t* src) {
  const int64_t d0 = (int64_t)blockIdx.x * (kBlock * kGatherV) + threadIdx.x;
  uint32_t k[kGatherV];
  bool ok[kGatherV];
#pragma unroll
  for (int v = 0; v < kGatherV; ++v) {
    const int64_t d = d0 + v * kBlock;
    ok[v] = d < in.n;
    k[v] = ok[v] ? src[d] : 0u;
  }
  gather_column(out.i1, (const int32_t*)in.i1, k, ok, d0);
  gather_column(out.i2, (const int32_t*)in.i2, k, ok, d0);
  gather_column(out.dx1, (const T*)in.dx1, k, ok, d0);
  gather_column(out.dx2, (const T*)in.dx2, k, ok, d0);
  gather_column(out.u1, (const T*)in.u1, k, ok, d0);
  gather_column(out.u2, (const T*)in.u2, k, ok, d0);
  gather_column(out.u3, (const T*)in.u3, k, ok, d0);
  if (in.phi) gather_column(out.phi, (const T*)in.phi, k, ok, d0);
  if (in.i1p) {
    gather_column(out.i1p, (const int32_t*)in.i1p, k, ok, d0);
    gather_column(out.i2p, (const int32_t*)in.i2p, k, ok, d0);
    gather_column(out.dx1p, (const T*)in.dx1p, k, ok, d0);
    gather_column(out.dx2p, (const T*)in.dx2p, k, ok, d0);
  }
  gather_column(const_cast<T*>(out.w), in.w, k, ok, d0);
  gather_column(out.tag, (const uint8_t*)in.tag, k, ok, d0);
}

// exclusive scan of uint32 in three passes: 1024 threads x 4 items per block
constexpr int kScanBlock = 1024;
constexpr int kScanItems = 4;
constexpr int kScanTile = kScanBlock * kScanItems;

__device__ __forceinline__ uint32_t block_exclusive_scan(uint32_t v, uint32_t* total) {
  __shared__ uint32_t warp_sums[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  uint32_t x = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
    if (lane >= o) x += y;
  }
  if (lane == 31) warp_sums[wid] = x;
  __syncthreads();
  if (wid == 0) {
    uint32_t s = warp_sums[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += y;
    }
    warp_sums[lane] = s;
  }
  __syncthreads();
  const uint32_t warp_off = wid ? warp_sums[wid - 1] : 0u;
  if (total) *total = warp_sums[31];
  __syncthreads();
  return warp_off + x - v;
}

__global__ void __launch_bounds__(kScanBlock) k_scan_local(uint32_t* data, uint32_t n, uint32_t* block_sums) {
  const uint32_t base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  uint32_t v[kScanItems], sum = 0;
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    v[j] = (base + j < n) ? data[base + j] : 0u;
    sum += v[j];
  }
  uint32_t total;
  uint32_t off = block_exclusive_scan(sum, &total);
#pragma unroll
  for (int j = 0; j < kScanItems; ++j) {
    if (base + j < n) data[base + j] = off;
    off += v[j];
  }
  if (threadIdx.x == 0) block_sums[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanBlock) k_scan_sums(uint32_t* block_sums, uint32_t nb) {
  uint32_t carry = 0;
  for (uint32_t start = 0; start < nb; start += kScanBlock) {
    const uint32_t i = start + threadIdx.x;
    const uint32_t v = (i < nb) ? block_sums[i] : 0u;
    uint32_t total;
    const uint32_t off = block_exclusive_scan(v, &total);
    if (i < nb) block_sums[i] = carry + off;
    carry += total;
  }
}

__global__ void __launch_bounds__(kScanBlock) k_scan_add(uint32_t* data, uint32_t n, const uint32_t* block_sums) {
  const uint32_t base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  const uint32_t add = block_sums[blockIdx.x];
#pragma unroll
  for (int j = 0; j < kScanItems; ++j)
    if (base + j < n) data[base + j] += add;
}

// Work items of the tiled step: (tile, first particle, count <= kChunk).  offsets[] is the scanned
// histogram (n_keys + 1 entries, the last two delimit the dead particles).
struct WorkItem {
  uint32_t tile, begin, count, pad;   // pad: 1 = dense item, served by k_step_lanes
};

__global__ void k_items_count(const uint32_t* offsets, uint32_t n_tiles, uint32_t* n_items_of_tile) {
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_tiles) return;
  const uint32_t cnt = offsets[(t + 1) * kTile * kTile] - offsets[t * kTile * kTile];
  n_items_of_tile[t] = (cnt + kChunk - 1) / kChunk;
}

// dense_min > 0: items of at least dense_min particles are marked (pad = 1) and listed in dense_idx for
// k_step_lanes (grpic_lanes.cuh); k_step_tiled then leaves them alone.  n_out: [0] items, [1] alive, [2] dense items
// ([2] zeroed by the caller).
__global__ void k_items_fill(const uint32_t* offsets, uint32_t n_tiles, const uint32_t* item_offset_of_tile,
                             WorkItem* items, uint32_t* n_out, uint32_t* dense_idx, uint32_t dense_min) {
  const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_tiles) return;
  const uint32_t b = offsets[t * kTile * kTile], e = offsets[(t + 1) * kTile * kTile];
  uint32_t k = item_offset_of_tile[t];
  for (uint32_t s = b; s < e; s += kChunk) {
    const uint32_t cnt = min((uint32_t)kChunk, e - s);
    const uint32_t dense = (dense_min > 0u && cnt >= dense_min) ? 1u : 0u;
    if (dense) dense_idx[atomicAdd(&n_out[2], 1u)] = k;
    items[k++] = WorkItem{t, s, cnt, dense};
  }
  if (t == n_tiles - 1) {
    n_out[0] = k;
    n_out[1] = e;
  }
}

}  // namespace grpic
