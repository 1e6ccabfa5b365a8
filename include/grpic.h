/*
 * grpic.h — C ABI of the B200-native per-particle GRPIC hot path.
 *
 * What is behind it: the per-particle step of the general-relativistic particle-in-cell
 * method of arxiv/paper_2511_17701 ("Entity II: General Relativistic Module") on a 2D
 * axisymmetric (r, theta) Kerr-Schild grid, as hand-written sm_100a CUDA kernels — and, around it,
 * the field-solver half of the same timestep (auxiliary fields, Faraday, Ampere, field boundary
 * conditions), so that the calls below close the PIC loop of Sec. 3.4.
 * "P:n" below = line n of the paper text; "R-Sk" = reading k of DESIGN.md.
 *
 * Two builds of one source export the SAME symbols:
 *     libgrpic_f32.so   grpic_real = float
 *     libgrpic_f64.so   grpic_real = double      (compile consumers with -DGRPIC_F64)
 * grpic_real_bytes() tells which one was loaded.
 *
 * Conventions
 *   - Every pointer inside grpic_particles / grpic_fields / grpic_current is CALLER-OWNED DEVICE
 *     memory (cudaMalloc'ed, or a torch CUDA tensor's data_ptr).  The *_host entry point is the one
 *     exception and says so.  The structs themselves live in host memory and are read during the call.
 *   - The library owns only its context (constants, counters, sort scratch, tile table).
 *   - Calls enqueue work on `cuda_stream` (a cudaStream_t passed as void*; NULL = legacy default
 *     stream) and return without synchronising, except grpic_counters, grpic_updates_total, grpic_sorted_alive,
 *     grpic_step_host, and the first grpic_sort of a context (scratch allocation).  grpic_step may use a side
 *     stream of the context next to `cuda_stream`, forked from it and joined back into it with events: to the caller
 *     everything is ordered on `cuda_stream`.
 *   - A context belongs to the CUDA device that was current at grpic_create; calls made with another device
 *     current return GRPIC_ESTATE.
 *   - Return value: GRPIC_OK (0) or a negative grpic_status; grpic_last_error(ctx) gives the text.
 *     Nothing aborts or throws.  There is no CPU fallback: without a CUDA device every compute
 *     call returns GRPIC_ECUDA.
 *   - Grid arrays (fields, currents): shape [n1 + 2*nghost][n2 + 2*nghost], i2 fastest, element
 *     (i1, i2) of the physical mesh at [(i1 + nghost)*(n2 + 2*nghost) + (i2 + nghost)].
 *     Yee locations (Eq. 40-41):
 *         D1(i+1/2, j)  D2(i, j+1/2)  D3(i, j)      B1(i, j+1/2)  B2(i+1/2, j)  B3(i+1/2, j+1/2)
 *     J^i sits where D^i sits.  Components are contravariant, code basis, code units.
 *     Ghost zones of the fields must be filled by the caller; the path reads one ghost
 *     layer.  Ghost zones of J are written raw (folding them back is field-side work).
 *   - Code coordinates: x1 in [0, n1) is radial with r = r_min * exp(x1 * ln(r_max/r_min)/n1)
 *     (App. A.3 with r0 = 0), x2 in [0, n2) is polar with theta = x2 * pi/n2; a position
 *     is (cell index i, displacement dx in [0,1)) per axis.  r_g = M = 1.  This is the default
 *     map, the one of the five benchmark configs; the other maps of App. A (uniform r, radial offset,
 *     polar stretch, flat space) are selected with grid.r_map and grpic_set_real (see there).
 */
#ifndef GRPIC_H_
#define GRPIC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#ifdef GRPIC_F64
typedef double grpic_real;
#else
typedef float grpic_real;
#endif

typedef enum {
  GRPIC_OK = 0,
  GRPIC_EINVAL = -1, /* bad argument (NULL pointer, n < 0, nghost < 1, ...)        */
  GRPIC_ENOMEM = -2, /* device or host allocation failed                           */
  GRPIC_ECUDA = -3,  /* CUDA runtime error or no device (text in grpic_last_error) */
  GRPIC_ESTATE = -4  /* call out of order (deposit before any push, ...)           */
} grpic_status;

typedef struct grpic_ctx grpic_ctx; /* opaque, library-owned */

/* The mesh: n1 = N_r, n2 = N_theta cells, nghost >= 1 ghost layers on every side. */
typedef struct {
  int32_t n1, n2, nghost;
  int32_t r_map; /* 1 = logarithmic r (quasi-spherical map of App. A.3; "r0", "h0" via grpic_set_real);
                    0 = uniform r (spherical Kerr-Schild of App. A.2: r = r_min + x1 (r_max - r_min)/n1) */
} grpic_grid;

/* One species, structure-of-arrays.
 * Columns of length >= n; slots with tag == 0 are dead and ignored by every call.
 * 16-byte alignment of every column is required (torch / cudaMalloc give 256). */
typedef struct {
  int64_t n;                   /* slots in use (alive + dead)                                   */
  int32_t *i1, *i2;            /* cell index                                     in/out         */
  grpic_real *dx1, *dx2;       /* displacement in [0,1)                          in/out         */
  grpic_real *u1, *u2, *u3;    /* covariant four-velocity, code basis            in/out         */
  grpic_real *phi;             /* out-of-plane angle (Eq. 30); may be NULL       in/out         */
  int32_t *i1_prev, *i2_prev;  /* position before the push: written by push,     read by deposit */
  grpic_real *dx1_prev, *dx2_prev;
  const grpic_real *weight;    /* macro-particle weight                          in             */
  uint8_t *tag;                /* 1 alive, 0 dead                                in/out         */
  double q_over_m;             /* charge/mass in code units; 0 skips the EM push        */
  double charge;               /* charge of one unit of weight, multiplies the deposit (Eq. 33) */
  int32_t massive;             /* 1: gamma = sqrt(1 + h^ij u_i u_j); 0: massless (Eq. 20), no EM push */
} grpic_particles;

typedef struct { const grpic_real *D1, *D2, *D3, *B1, *B2, *B3; } grpic_fields;
typedef struct { grpic_real *J1, *J2, *J3; } grpic_current; /* ACCUMULATED into; caller zeroes */

/* sizeof(grpic_real) of the loaded build: 4 or 8. */
int grpic_real_bytes(void);

/* Create a context for one mesh and one Kerr spin a (|a| <= 1), radial extent [r_min, r_max]
 * in units of r_g (north_star: grpic_create(grid, a, r_min, r_max); metric of App. A.3).
 * Defaults: n_iter = 10, small_angle = 1e-5 (SMALL_ANGLE_GR).
 * Errors: EINVAL (NULL, n1/n2 < 1, nghost < 1, r_map not 0 or 1, r_min <= 0 or >= r_max), ECUDA, ENOMEM. */
int grpic_create(const grpic_grid* grid, double a, double r_min, double r_max, grpic_ctx** out);
int grpic_destroy(grpic_ctx* ctx);

/* "n_iter": fixed iteration count of the two midpoint integrators, 1..64.
 * "early_exit": 1 (default) leaves a fixed-point loop as soon as an iterate repeats the previous one bit
 *              for bit — every later iterate would be that same value, so the result IS the one of
 *              n_iter iterations; 0 always executes all n_iter (used by the test that proves this).
 * "tile_path": 1 (default) lets grpic_step use the shared-memory tile kernels after a grpic_sort;
 *              0 forces the direct kernel (global gathers and atomics).
 * "lanes_path": 1 (default) sends the dense work items of a sorted species (at least "dense_min" particles of one
 *              16 x 16-cell tile, default 2048, range 4..16384; read at the next grpic_sort) to k_step_lanes: one run of sorted
 *              particles per lane, current accumulated in lane-private shared-memory windows, columns moved as 16-byte
 *              blocks - this needs every particle column 16-byte aligned, otherwise (or with 0) all items stay with
 *              the warp-by-warp tile kernel.  Same results up to the order of the J additions.
 * "overlap":   1 (default) runs the small kernels of grpic_step (sparse items, slots behind the sorted range) on the side
 *              stream beside k_step_lanes; 0 keeps everything on `cuda_stream`.
 * "tma": 1 (default) stages the tile's field stencil with TMA; 0 uses plain cooperative loads (also the
 *        automatic choice when a field array is not 16-byte aligned or (n2 + 2 nghost)*sizeof(real) % 16 != 0).
 * "host_chunk": particles per chunk of grpic_step_host, 2^10..2^26 (default 2^22; three chunks in flight). */
int grpic_set_int(grpic_ctx* ctx, const char* key, int64_t value);
/* "small_angle": theta used in any metric evaluation is clamped to [eps, pi - eps] (R-S9).
 * "r0", "h0":    the remaining parameters of the quasi-spherical map of App. A.3, both 0 by default:
 *                xi = log(r - r0) uniform in x1 (r0 < r_min; r_min, r_max keep their meaning), and
 *                theta = eta + 2 h0 eta (pi - 2 eta)(pi - eta)/pi^2 with eta = x2*pi/n2 (-0.5 < h0 < 1).
 * "mass":        M in units of r_g, default 1.  0 together with a = 0 gives the flat spherical metric
 *                kerr_schild_0 of App. A.1 that the paper uses for its SR-EM test.
 *                With any of these off its default every call runs the same kernels instantiated with the general coordinate
 *                class (plain evaluation of the map at every point instead of the default map's shortcuts).
 * "sort_lookahead": L in [0, 64] steps (default 0).  With L > 0 grpic_sort / grpic_sort_into order the particles
 *                by the cell each is PREDICTED to occupy L steps of the last dt ahead (ballistic:
 *                dx^i/dt = alpha h^ij u_j / gamma - beta^i of Eq. 28 at its present place, in FP32) instead of its present
 *                cell.  An ordering heuristic only: any order is a correct sort result and grpic_step gives the same
 *                results on it (a particle outside its tile's shared-memory window takes the global path).  With
 *                L = half the sort interval the particles of a warp are closest together in the MIDDLE of the interval,
 *                which the warp-level deposit aggregation rewards (config 4: -3 % per sort interval).  No effect before the
 *                first push on the context (no dt yet). */
int grpic_set_real(grpic_ctx* ctx, const char* key, double value);

/* Steps 1-11 of Sec. 3.1 for every alive particle, then the particle boundary
 * conditions: save previous position; interpolate D, B (R-S4); tetrad-frame Boris half
 * push (Eq. 19, R-S5); geodesic momentum push (Eq. 26-27); second half push; geodesic coordinate
 * push (Eq. 28-29); phi (Eq. 30); renormalise (i, dx); reflect at the axes; tag = 0 for i1 < 0
 * (inside the horizon) or i1 >= n1.  `fields` may be NULL iff q_over_m == 0 or massive == 0.
 * Remembers dt for grpic_deposit.  Errors: EINVAL, ECUDA. */
int grpic_interp_push(grpic_ctx* ctx, grpic_particles* p, const grpic_fields* fields, double dt,
                      void* cuda_stream);

/* Charge-conserving conformal current deposit (Sec. 3.2, Eq. 32-36; scheme R-S10) from
 * (i*_prev, dx*_prev) to (i*, dx*) of every alive particle, with the dt of the last push on this
 * context.  J += ; a no-op if charge == 0.  A particle that moved more than one cell along an axis
 * is skipped and counted (n_overstep).  Errors: EINVAL, ESTATE (no push yet), ECUDA. */
int grpic_deposit(grpic_ctx* ctx, const grpic_particles* p, grpic_current* J, void* cuda_stream);

/* Fused grpic_interp_push + grpic_deposit in one kernel: the previous position (step 1) stays
 * in registers.  It is also written to the four *_prev columns when they are given (so that a later
 * grpic_deposit / diagnostics see it); all four may be NULL, and then it is not stored at all.  Same
 * results as the two calls up to the order of the J additions.  J may be NULL iff charge == 0. */
int grpic_step(grpic_ctx* ctx, grpic_particles* p, const grpic_fields* fields, grpic_current* J,
               double dt, void* cuda_stream);

/* Counting sort of all columns by tile-major cell key (not in the paper; north_star names it; R-S9):
 *     key = ((i1/T * ceil(n2/T) + i2/T) * T + i1%T) * T + i2%T,  T = grpic_tile_size(),
 * of the present cell (i1, i2), or of the predicted cell when "sort_lookahead" > 0,
 * dead particles after all alive ones.  In place from the caller's view (library scratch inside).
 * Any order within one key is a correct result.  Builds the tile table that grpic_step's
 * shared-memory path uses for this species (keyed by the address of p->i1).  Enqueues and returns: the number of alive
 * particles stays on the device (grpic_sorted_alive fetches it); only the first call on a context, or a call with more
 * particles than any before, synchronises to (re)allocate scratch.
 * Errors: EINVAL, ENOMEM, ECUDA. */
int grpic_sort(grpic_ctx* ctx, grpic_particles* p, void* cuda_stream);

/* The same sort out of place: reads the columns of `src` (left unchanged) and writes them in sorted order
 * into the columns of `dst` — same n, same optional columns, no column shared between the two.  Saves the
 * library-side snapshot of every column that the in-place call needs (a caller that keeps two column sets
 * and swaps them after each sort moves every byte once instead of twice).  The tile table is built for
 * `dst` (keyed by the address of dst->i1).  In both calls phi and the four *_prev columns are optional
 * (*_prev: all or none).  Errors: EINVAL, ENOMEM, ECUDA. */
int grpic_sort_into(grpic_ctx* ctx, const grpic_particles* src, grpic_particles* dst, void* cuda_stream);
int grpic_tile_size(void);

/* Compaction / injection support.  After grpic_sort the alive particles of the species occupy the slots
 * [0, n_alive) and the dead ones the rest; this call returns that n_alive, read back from the device (it synchronises the
 * stream of that sort, once per sort) (the caller may set p->n = n_alive to drop the
 * dead slots, or write new particles into slots >= n_alive with tag = 1, or append beyond p->n and raise p->n).
 * grpic_step pushes such slots through the direct kernel until the next grpic_sort, whatever was sorted before.
 * Errors: EINVAL, ESTATE (species never sorted on this context). */
int grpic_sorted_alive(grpic_ctx* ctx, const grpic_particles* p, int64_t* n_alive);

/* Drop the tile table the last grpic_sort built for this species (found by the address of p->i1): call it before the
 * storage of a sorted species is freed or handed to another species, so that a recycled address cannot meet a stale
 * table (results would still be right - every particle is tested against its tile's window - but the step would take the
 * slow global path).  The library keeps at most 64 tables per context and evicts the one sorted longest ago.
 * Synchronises the device (the table may still be in use).  Errors: EINVAL, ESTATE. */
int grpic_forget(grpic_ctx* ctx, const grpic_particles* p);

/* Counters of the most recent push/step (alive after it, absorbed inside, absorbed outside) and
 * of the most recent deposit/step (n_overstep).  Synchronises `cuda_stream`. Any pointer may be NULL. */
int grpic_counters(grpic_ctx* ctx, int64_t* n_alive, int64_t* n_absorbed_in, int64_t* n_absorbed_out,
                   int64_t* n_overstep, void* cuda_stream);

/* Number of particle updates (alive particles pushed) by all push/step calls since grpic_create:
 * the numerator of the throughput metric.  Synchronises `cuda_stream`. */
int grpic_updates_total(grpic_ctx* ctx, int64_t* n_updates, void* cuda_stream);

/* Throughput probes: the measured denominators of the ALU roofline (bench.py --peaks and every bench line).  Enqueues ONE
 * launch of a register-only kernel on `cuda_stream` (1184 blocks x 256 threads, 8 independent chains per thread) and
 * returns in *ops the operations that launch executes; the caller times it with CUDA events.
 *   "ffma": FP32 fused multiply-adds, *ops in flop (2 per FMA);  "dfma": FP64 likewise;
 *   "mufu": rsqrt.approx.f32 (special-function unit), *ops in thread operations;
 *   "smem_rmw": LDS + FADD + STS on lane-private shared words (the read-modify-write of k_step_lanes' windows).
 * Errors: EINVAL, ECUDA. */
int grpic_probe(grpic_ctx* ctx, const char* what, int64_t iters, int64_t* ops, void* cuda_stream);

/* ---- Field-solver half of the step (Sec. 3.3).  Grid kernels; same array layout; device pointers. ----
 * The caller sequences them and the time levels (Sec. 3.4) and fills the ghost ROWS i < 0, i >= n1 of the inputs
 * (P:461-467); ghost columns beyond the axes are not read.  Rows written: every row whose x1-stencil lies inside the
 * arrays (aux: array rows 1 .. rows-2; Faraday/Ampere: array rows 2 .. rows-3; with nghost = 2 that is the whole mesh).
 * The metric at every Yee location is evaluated in FP64 in both builds. */
typedef struct { grpic_real *F1, *F2, *F3; } grpic_vec3;

/* Auxiliary fields (Eq. 38, 42-44): E_i = alpha h_ij D^j + e_ijk beta^j B^k at the D^i locations and
 * H_i = alpha h_ij B^j - e_ijk beta^j D^k at the B^i locations; components at other Yee locations are brought over by
 * the two-point volume-weighted average along x1 (Eq. 43) written with sqrt(h)/sin(theta).
 * E or H may be NULL (only the other is computed).  Errors: EINVAL, ECUDA. */
int grpic_aux_fields(grpic_ctx* ctx, const grpic_fields* em, grpic_vec3* E, grpic_vec3* H, void* cuda_stream);

/* Faraday (Eq. 40): B^i -= dt e^{ijk} d_j E_k / sqrt(h), B^2 on the axes untouched. */
int grpic_faraday(grpic_ctx* ctx, grpic_vec3* B, const grpic_vec3* E, double dt, void* cuda_stream);

/* Ampere (Eq. 41): D^i += dt (e^{ijk} d_j H_k - k_J J^i)/sqrt(h) with the deposited conformal currents J (may be NULL);
 * k_J = 4 pi unless changed with grpic_set_real("k_J").  D^3 on the axes untouched; D^1 on the axes by the integral
 * form Eq. 45 with the polar area of App. A. */
int grpic_ampere(grpic_ctx* ctx, grpic_vec3* D, const grpic_vec3* H, const grpic_current* J, double dt, void* cuda_stream);

/* Field boundary conditions (Sec. 3.3.3), in place on D^i and B^i: the ghost columns beyond the two polar
 * axes by reflection (r- and phi-components even, theta-components odd; Fig. 1), B^2 = D^3 = 0 on the axes, and,
 * if n_const >= 0, the constant layer inside the horizon: rows i1 in [-nghost, n_const] take the values of row
 * n_const + 1 (n_const = number of current-filter passes).  The absorbing layer at the outer edge is
 * grpic_field_match.  Errors: EINVAL, ECUDA. */
int grpic_field_bc(grpic_ctx* ctx, grpic_vec3* D, grpic_vec3* B, int32_t n_const, void* cuda_stream);

/* Absorbing layer at the outer radial boundary, in place on D^i and B^i: "the fields are matched to their initial
 * values using an absorbing layer", "we smoothly match the field components with the analytic solution"
 * (P:644).  The paper defers the profile to paper I; reading R-F6 of DESIGN.md: for r_abs < r
 *     F <- F_target + s (F - F_target),   s = tanh(4 (r_max - r) / (r_max - r_abs)),  s = 0 for r >= r_max,
 * with r the radius of each component's own Yee location; rows with r <= r_abs are not touched.  D_target, B_target:
 * device arrays of the grid layout (the initial or analytic fields), read only.  r_abs in [r_min, r_max).
 * Errors: EINVAL, ECUDA. */
int grpic_field_match(grpic_ctx* ctx, grpic_vec3* D, grpic_vec3* B, const grpic_vec3* D_target, const grpic_vec3* B_target,
                      double r_abs, void* cuda_stream);

/* Current filter ("n_f passes of a digital filter"; the paper defers its form to paper I — reading R-F5 of
 * DESIGN.md): n_passes of the binomial smoothing [1 2 1]/4 along x2 and along x1, in place on J, each component on its
 * own Yee lattice; mirror samples with the component's parity beyond the polar axes; the first and last array rows are
 * not smoothed along x1.  Errors: EINVAL, ENOMEM (scratch), ECUDA. */
int grpic_filter_current(grpic_ctx* ctx, grpic_current* J, int32_t n_passes, void* cuda_stream);

/* Field side of one PIC timestep (Sec. 3.4), built from the three operations above.  The state holds
 * (n-3/2)B, (n-1/2)B, (n-1)D, (n)D; all arrays caller-owned device memory; library scratch: 12 grid arrays.
 *   grpic_fields_prepare  step 2, Eq. 46-48: B_n <- (n)B, the magnetic field aligned in time with (n)D for the push
 *                         (grpic_interp_push / grpic_step then take D = state.D, B = B_n).
 *   grpic_fields_advance  steps 5-7, Eq. 51-56, after the deposit of (n+1/2)J: (n)J = ((n-1/2)J + (n+1/2)J)/2;
 *                         (n)E,(n)H; main Faraday (n-1/2)B -> (n+1/2)B; auxiliary Ampere (n-1/2)D -> (n+1/2)D with
 *                         (n)H,(n)J; (n+1/2)H; final Ampere (n)D -> (n+1)D with (n+1/2)H,(n+1/2)J.
 *                         On return the state holds (n-1/2)B, (n+1/2)B, (n)D, (n+1)D in B_prev, B, D_prev, D.
 *                         J_prev = (n-1/2)J and J = (n+1/2)J, or both NULL (vacuum).
 * Errors: EINVAL, ENOMEM (scratch), ECUDA. */
typedef struct { grpic_vec3 B_prev, B, D_prev, D; } grpic_field_state;
int grpic_fields_prepare(grpic_ctx* ctx, const grpic_field_state* s, grpic_vec3* B_n, double dt, void* cuda_stream);
int grpic_fields_advance(grpic_ctx* ctx, grpic_field_state* s, const grpic_vec3* B_n, const grpic_current* J_prev,
                         const grpic_current* J, double dt, void* cuda_stream);

/* End-to-end convenience: every pointer in p, fields and J is HOST memory (pinned or pageable).
 * Copies fields and particle columns to library-owned device buffers in chunks, runs the fused step
 * chunk by chunk (three chunks in flight on three streams: upload, compute, download), and copies the
 * particle columns back; J_host += (the host values are uploaded, the deposit adds to them on the device, the
 * sums come back).  The four *_prev columns of p_host may all be NULL:
 * the fused step keeps the previous position on the device and nothing is copied back for them.
 * Synchronous.  Bytes moved are reported through
 * h2d_bytes / d2h_bytes (may be NULL).  Errors as grpic_step, plus ENOMEM. */
int grpic_step_host(grpic_ctx* ctx, grpic_particles* p_host, const grpic_fields* fields_host,
                    grpic_current* J_host, double dt, int64_t* h2d_bytes, int64_t* d2h_bytes);

/* Text of the last error on this context (or of the last failed grpic_create if ctx == NULL).
 * Owned by the library, valid until the next call. */
const char* grpic_last_error(grpic_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* GRPIC_H_ */
