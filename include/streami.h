/* include/streami.h -- C ABI of the B200-native particle-update library
 * (libstreami_b200.so, sources in paper_2606_02627_b200/csrc/).
 *
 * What it computes: the particle-update step of field-line tracing as described in
 * "Streami: An MPI Data-Parallel Library to Compute Field Lines on GPUs"
 * (arxiv/paper_2606_02627; citations are /root/reference/PAPER.md:<line>):
 *   - update() kernel, one RK4 step per particle with four field.sample() calls and
 *     "a failed sample ends the particle"            Listing 1
 *   - VecField::sample() / destinationID(), macrocell + halo
 *   - structured field = array of float3 voxels, sampled by offset computation
 *   - Tracer::step()/trace() loop, streakline batches per step, fields[simStep]
 *                                                    Listing 2
 *   - particle = position + unique id
 *   - emitOutgoing / forward until no particle is active anywhere
 * Where the paper is silent (trilinear filter, linear interpolation in time, |v| floor,
 * adaptive Dormand-Prince 5(4), capacity/stride recording) BASELINE.json binds and the fp32
 * formula sheet A1-A9 (restated in DESIGN.md section 3) fixes every operation.
 *
 * Conventions
 *   - "device" pointers are CUDA device memory owned by the caller (e.g. torch tensors);
 *     "host" pointers are ordinary host memory.  No torch types cross this boundary.
 *   - Every call returns int: 0 ok, negative = error (STREAMI_E_*).  Nothing is printed, no
 *     exception crosses the ABI.  Bad *particles* are not errors (a seed outside the domain gets
 *     status OUT_OF_DOMAIN, 0 steps, 0 vertices).
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Work
 *     is enqueued on it; outputs are valid after the caller synchronises that stream, unless a
 *     function says that it synchronises the stream itself.  No call synchronises the device.
 *   - All per-particle outputs are indexed by particle id (= seed index; streaklines:
 *     release*m + point), so they do not depend on scheduling, sorting or queue order.
 *   - There is no CPU fallback: without a CUDA device every compute call returns STREAMI_E_CUDA.
 */
#ifndef STREAMI_H
#define STREAMI_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

/* error codes */
#define STREAMI_OK            0
#define STREAMI_E_INVALID    (-1)  /* null pointer, dim < 2, spacing <= 0 or non-finite, nslices < 1,
                                      capacity == 0, stride == 0, h <= 0, h_min > h_max, ... */
#define STREAMI_E_NOMEM      (-2)  /* out of device memory */
#define STREAMI_E_CUDA       (-3)  /* CUDA error; text behind streami_error_string(-3) */
#define STREAMI_E_TRUNCATED  (-4)  /* hand-off log or round table overflowed; results still valid */
#define STREAMI_E_TOO_LARGE  (-5)  /* streami_trace_streamlines_noalloc: more seeds than its static scratch holds */

/* termination reasons (A5) written to out_status */
#define STREAMI_ALIVE          0u  /* never final */
#define STREAMI_OUT_OF_DOMAIN  1u  /* a stage sample or the new position left the domain (Listing 1's return) */
#define STREAMI_MAX_STEPS      2u  /* reached max_steps (streaklines: alive at the end) */
#define STREAMI_STAGNANT       3u  /* |v(p)| < vmin */
#define STREAMI_HALO_MISS      4u  /* bricks only: a stage point left the brick's stored box */

/* field layouts (layout_hint of streami_field_create*, reported by streami_field_info) */
#define STREAMI_LAYOUT_AUTO    0   /* library chooses the FASTEST layout whose library-owned copy fits HALF of the
                                      device memory that is free at create time: steady
                                      fields CELL (10.7x the packed size), else XYQUAD (5.3x), else XPAIR (2.7x);
                                      unsteady fields XPAIR; falls back to the next smaller layout, in the end to
                                      the caller's array in place, instead of failing with NOMEM.  The copy is
                                      the price of speed: streami_field_info reports the layout chosen and the
                                      bytes it took.  A caller that cannot spare the memory passes PACKED3 (no
                                      copy at all) or FLOAT4 (1.3x) explicitly. */
#define STREAMI_LAYOUT_PACKED3 1   /* use the caller's packed float3 array in place (the paper's layout) */
#define STREAMI_LAYOUT_FLOAT4  2   /* library-owned copy padded to 16 B per vertex */
#define STREAMI_LAYOUT_XPAIR   3   /* library-owned copy, 32 B per vertex: V[x] and V[x+1] - V[x]: one
                                      aligned sector per trilinear row */
#define STREAMI_LAYOUT_XYQUAD  5   /* library-owned copy, 64 B per vertex: the XPAIR rows (x, y) and (x, y+1):
                                      a cell is two aligned 64-byte pieces (4x the packed size) */
#define STREAMI_LAYOUT_SOA     6   /* library-owned copy, three component planes of fp32 (12 B per vertex); a comparison
                                      layout: measured and rejected, kept selectable */
#define STREAMI_LAYOUT_TEX     7   /* library-owned float4 copy read through a texture object in POINT mode (tex1Dfetch,
                                      lerps in registers); comparison layout, measured and rejected; INVALID for
                                      stores of more texels than a linear texture holds */
#define STREAMI_LAYOUT_CELL    4   /* library-owned copy, 128 B per CELL: its 8 corner vertices in one
                                      aligned L2 line (10.7x the packed size) */

typedef struct streami_field_s* streami_field;   /* opaque host-side handle (D2/D3) */

typedef struct {                 /* all fp32 scalars are used bit-for-bit */
  int      integrator;           /* 0 = RK4 fixed step (Listing 1), 1 = Dormand-Prince 5(4) adaptive (A8) */
  float    h;                    /* RK4 step; DP5(4) initial step */
  float    h_min, h_max;         /* DP5(4) only */
  float    atol, rtol;           /* DP5(4) only */
  unsigned max_steps;            /* accepted steps per particle (ignored by streaklines) */
  float    vmin;                 /* terminate when |v(p)| < vmin (0 disables) */
  float    t0;                   /* time of step 0 (unsteady fields) */
  int      time_mode;            /* 0 = linear between slices, 1 = hold floor slice */
  unsigned capacity;             /* vertex slots per particle (A6) */
  unsigned stride;               /* record vertex k iff k % stride == 0 and k/stride < capacity */
  /* optional extra outputs, device pointers, may be NULL: */
  unsigned* out_steps;           /* [n] accepted steps */
  unsigned* out_status;          /* [n] termination reason */
  float*    out_final;           /* [3][n] last inside position (SoA) */
  unsigned long long* out_totals;/* [4] attempted steps, accepted steps, field samples, hand-offs;
                                    overwritten (not accumulated) by each call */
} streami_params;

/* Create a field over a caller-owned packed array ("a CUDA global memory array
 * for the voxels"): dev_ptr = [nslices][Nz][Ny][Nx][3] fp32, x fastest, vertex-centred (A1).
 * dev_ptr is BORROWED for the life of the handle and never written.  With layout_hint other
 * than PACKED3 the library makes its own repacked copy (owned by the handle, freed by
 * _destroy); the repack runs on the legacy default stream and is complete on return.
 * slice_dt is the time between slices (ignored when nslices == 1).
 * Errors: INVALID (null, dims < 2, spacing <= 0 or non-finite, nslices < 1, slice_dt <= 0,
 * more than 2^32-1 vertices per slice, unknown layout), NOMEM, CUDA. */
int streami_field_create(const int dims[3], const float origin[3], const float spacing[3],
                         int nslices, float slice_dt, const float* dev_ptr, int layout_hint,
                         streami_field* out);

/* Create a brick-decomposed steady field (macrocells + halo; A9).  The global
 * grid global_dims is cut by brick_grid = (nbx, nby, nbz) into bricks of B_a = N_a / nb_a cells
 * (the last brick of an axis takes the remainder).  Brick b = (bz*nby + by)*nbx + bx STORES the
 * vertex box lo_a = max(B_a*b_a - ghost, 0) .. hi_a = min(B_a*(b_a+1) + ghost, N_a-1) (hi_a =
 * N_a-1 for the last brick) as its own packed float3 array brick_dev_ptrs[b] (host array of
 * device pointers), the way each MPI rank of the paper holds its partition.  Same ownership
 * and layout rules as streami_field_create, per brick.  ghost >= 1. */
int streami_field_create_bricked(const int global_dims[3], const float origin[3],
                                 const float spacing[3], const int brick_grid[3], int ghost_cells,
                                 const float* const* brick_dev_ptrs, int layout_hint,
                                 streami_field* out);

int streami_field_destroy(streami_field f);

/* Layout actually used and device bytes owned by the handle (0 for PACKED3). */
int streami_field_info(streami_field f, int* layout, size_t* owned_bytes);

/* a2-a4 alone: sample the field at n device points [n][3] at time t (A2/A3).
 * out_v [n][3] (zero where not ok), out_rc [n] = 0 ok / OUT_OF_DOMAIN.  Monolithic fields only. */
int streami_sample(streami_field f, const float* points, size_t n, float t, int time_mode,
                   float* out_v, unsigned* out_rc, void* cuda_stream);

/* Streamlines (Tracer::trace() in Streamlines mode; A4-A6, A8).
 * seeds [n][3] device AoS.  out_vertices [3][n][capacity] device SoA planes, slot k/stride of
 * particle id at c*n*capacity + id*capacity + k/stride; slots beyond out_counts[id] are left
 * untouched.  out_counts [n] device = stored vertices per particle.  out_vertices may be NULL
 * (nothing recorded, out_counts still written).  Asynchronous on cuda_stream; scratch memory
 * is taken from the stream-ordered allocator.  n == 0 is ok.  Monolithic fields only.
 * Errors: INVALID (null field/seeds/params/out_counts, capacity == 0, stride == 0, h <= 0 or
 * non-finite, DP5: h_min <= 0, h_min > h_max, atol/rtol < 0), NOMEM, CUDA. */
int streami_trace_streamlines(streami_field f, const float* seeds, size_t n,
                              const streami_params* params, float* out_vertices,
                              unsigned* out_counts, void* cuda_stream);

/* The same call for callers that cannot allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): identical arguments, identical outputs (the same kernels run), but ALL
 * scratch -- the persistent kernel's work counter and, from 65,536 seeds on, the Morton presort's histogram, keys,
 * permutation and gathered seeds -- lives in one static device array of the library (7,341,312 bytes, held by
 * every GPU that loads the library until exit) instead of coming from the stream-ordered allocator.  The call
 * makes no cudaMalloc / cudaMallocAsync / cudaFree and creates no events or streams.  Limits and rules:
 *   - n <= STREAMI_NOALLOC_MAX_SEEDS, else STREAMI_E_TOO_LARGE (nothing is enqueued);
 *   - monolithic fields; one launch to the end (options "segment_steps", "queue_steps" and "kernel_timing"
 *     are ignored);
 *   - every call on a device shares the array: the call clears what must start at zero itself, on cuda_stream,
 *     but two calls that OVERLAP on the GPU (different streams without an ordering between them) race on it and
 *     give undefined results.  Calls on one stream, or ordered by events, are fine;
 *   - the first call on a device resolves the array's device address (cudaGetSymbolAddress, no allocation); make
 *     one call per device before capturing a graph.
 * Asynchronous on cuda_stream.  Errors: as streami_trace_streamlines, plus TOO_LARGE. */
#define STREAMI_NOALLOC_MAX_SEEDS 262144
int streami_trace_streamlines_noalloc(streami_field f, const float* seeds, size_t n,
                                      const streami_params* params, float* out_vertices,
                                      unsigned* out_counts, void* cuda_stream);

/* The same call with HOST buffers: seeds, out_vertices, out_counts and the optional outputs in
 * params are host pointers (pinned memory makes the copies faster but is not required).  Copies
 * host->device, traces, copies device->host and synchronises cuda_stream before returning. */
int streami_trace_streamlines_host(streami_field f, const float* seeds, size_t n,
                                   const streami_params* params, float* out_vertices,
                                   unsigned* out_counts, void* cuda_stream);

/* Streaklines (Listing 2; A7).  points [m][3] device.  Particle (i, j) is
 * released at point i at global step j and steps at global indices j..nsteps-1 with
 * t_s = t0 + (float)s*h (RK4 only; params->integrator must be 0; max_steps, capacity, stride are
 * ignored).  out_vertices [3][nsteps][m] device, release-major: slot (j, i) = final position of
 * particle id = j*m + i (its last inside position if it died).  out_counts [m] = particles of
 * point i alive at the end (status MAX_STEPS).  params->out_steps/out_status are [nsteps*m].
 * Asynchronous on cuda_stream. */
int streami_trace_streaklines(streami_field f, const float* points, size_t m, unsigned nsteps,
                              const streami_params* params, float* out_vertices,
                              unsigned* out_counts, void* cuda_stream);

/* Per-destination partition of seeds (A9: Q_0[b] = the seeds owned by brick b; the distribution step of a
 * data-parallel run, where every rank receives the particles of its macrocell).
 * out_perm [n] (device): the seed indices ordered by (owner brick, Morton code inside the brick) -- the same
 * two-level counting sort streami_brick_advect applies to every round's hand-off queue, so that the work
 * of a round is ONE contiguous segment per destination brick (the "send buffer" of that destination).
 * out_offsets [nbricks + 1] (device): segment b is out_perm[out_offsets[b] .. out_offsets[b+1]).  Seeds
 * outside the domain are listed with brick 0.  Order inside a (brick, block) bin is unspecified.
 * Asynchronous on cuda_stream.  Errors: INVALID (null, not a bricked field, n >= 2^32), NOMEM, CUDA. */
int streami_partition_seeds(streami_field bricked, const float* seeds, size_t n, unsigned* out_perm,
                            unsigned long long* out_offsets, void* cuda_stream);

/* Brick advection with hand-off (P1/K1/K3/K4 of SURVEY.md; A9).
 * f must come from streami_field_create_bricked; RK4 or DP5(4).  In round r every particle queued for
 * brick b is advected inside b until it ends or its new position is owned by another brick; it
 * is then appended to that brick's queue for round r+1 (the device-side stand-in for
 * emitOutgoing + the all-to-all forward).  Rounds run until no particle is queued anywhere.
 * Outputs as streami_trace_streamlines, plus (all optional, device unless noted):
 *   out_round_counts [max_rounds][nbricks]: |Q_r[b]| (rows beyond the executed rounds untouched)
 *   out_handoff_log  [log_capacity]: one entry (round+1)<<48 | dest<<32 | id per hand-off, in
 *                    unspecified order; out_log_count (device, 1 x u64) = hand-offs in total
 *   out_nrounds      HOST pointer: rounds executed.
 * out_nrounds counts launches: A9's rounds when the round table or the log is requested (or option
 * "brick_round_steps" = -1); otherwise the library may also cut a round after a step budget (option
 * "brick_round_steps": 0 = automatic, k > 0 = k steps per round; k = 1 is the paper's one-step
 * schedule), which changes no per-particle result.
 * This call synchronises cuda_stream once per round (it reads the live count) and before
 * returning.  Returns STREAMI_E_TRUNCATED if the log or the round table overflowed (all other
 * results are still valid). */
int streami_brick_advect(streami_field f, const float* seeds, size_t n,
                         const streami_params* params, float* out_vertices, unsigned* out_counts,
                         unsigned* out_round_counts, unsigned max_rounds,
                         unsigned long long* out_handoff_log, size_t log_capacity,
                         unsigned long long* out_log_count, unsigned* out_nrounds,
                         void* cuda_stream);

/* Vector fields on hexahedral meshes -- the paper's other field type ("unstructured meshes", cell
 * location + interpolation), restricted to the element type of its own
 * experiment (a structured grid re-expressed as hexahedra).  Formula sheet U1-U4:
 * cell c has corners H[c][l], l = dx + 2 dy + 4 dz, at reference coordinates (dx, dy, dz); a point
 * is located through a uniform bin grid nb over the box lo..hi as the first (lowest-numbered) cell
 * listed in its bin whose inverse isoparametric map (Newton from the centre, at most 6 steps) converges to
 * reference coordinates inside the unit cube (+- 2e-5); the value is the trilinear combination of
 * the corner values at those coordinates.
 * _create_hex: X [nv][3], V [nv][3], H [nc][8] are HOST arrays (consumed: the handle owns a device
 * copy in a per-cell layout and the bin lists, built here); errors: INVALID (null, empty, index
 * out of range, empty box, more than 2^32-1 list entries), NOMEM, CUDA.
 * _sample: points [n][3] device -> out_v [n][3] (zero where no cell is found), out_cell [n] i64
 * (-1 = outside; may be NULL).  _trace_streamlines: as streami_trace_streamlines (RK4 only;
 * out_vertices may be NULL; OUT_OF_DOMAIN = no cell contains the point). */
typedef struct streami_mesh_s* streami_mesh;
int streami_mesh_create_hex(size_t nv, size_t nc, const float* X, const float* V, const unsigned* H,
                            const float lo[3], const float hi[3], const int nb[3], streami_mesh* out);
int streami_mesh_destroy(streami_mesh m);
/* Host-only helpers (no device work).  _reorder_vtk_hex: H_vtk [nc][8] in VTK_HEXAHEDRON node order (0-3 the bottom
 * face counter-clockwise, 4-7 the top face above them) -> H_out [nc][8] in the corner order of this library
 * (l = dx + 2 dy + 4 dz); H_out may be H_vtk.  _check_hex: counts the cells whose Jacobian determinant at the cell
 * centre or at one of the 8 corners is not positive (inverted, degenerate or wrongly ordered cells: U3's Newton iteration does not converge in
 * them and their points report OUT_OF_DOMAIN) or that name a vertex >= nv; *out_first_bad = the first such cell or -1
 * (may be NULL).  Call it before _create_hex when the mesh comes from elsewhere.  Errors: INVALID (null). */
int streami_mesh_reorder_vtk_hex(size_t nc, const unsigned* H_vtk, unsigned* H_out);
int streami_mesh_check_hex(size_t nv, size_t nc, const float* X, const unsigned* H, unsigned long long* out_bad,
                           long long* out_first_bad);
int streami_mesh_sample(streami_mesh m, const float* points, size_t n, float* out_v, long long* out_cell,
                        void* cuda_stream);
int streami_mesh_trace_streamlines(streami_mesh m, const float* seeds, size_t n, const streami_params* params,
                                   float* out_vertices, unsigned* out_counts, void* cuda_stream);
/* As streami_trace_streamlines_lines_host (HOST seeds in, HOST polylines out, batched and overlapped
 * in the same way), on a mesh. */
int streami_mesh_trace_streamlines_lines_host(streami_mesh m, const float* seeds, size_t n,
                                              const streami_params* params, unsigned long long* out_offsets,
                                              float* out_points, unsigned long long max_points,
                                              unsigned long long* out_total, void* cuda_stream);

/* Seed generation on a control shape (the paper's convenience kernels: "uniformly distributed seed
 * points given simple control shapes such as planes or lines").  The shape is
 * origin + u*edge_u + v*edge_v + w*edge_w, (u,v,w) in [0,1)^3, sampled nu x nv x nw times (line:
 * nv = nw = 1; plane: nw = 1); seed s = (k*nv + j)*nu + i goes to out_seeds [nu*nv*nw][3] (device,
 * the seeds argument of the trace calls).  mode 0 = lattice at the sub-cell centres
 * ((i+0.5)/nu, ...), mode 1 = uniformly random from a counter-based generator keyed by rng_seed
 * (the same seeds for the same key on any launch geometry).  edge pointers are HOST arrays.
 * Asynchronous on cuda_stream.  Errors: INVALID (null, unknown mode, more than 2^32-1 seeds). */
int streami_seed_shape(const float origin[3], const float edge_u[3], const float edge_v[3],
                       const float edge_w[3], unsigned nu, unsigned nv, unsigned nw, int mode,
                       unsigned long long rng_seed, float* out_seeds, void* cuda_stream);

/* Step-synchronous streaklines: Tracer::step() of Listing 2 ("one advection step
 * ... then a new batch of particles").  _begin binds the rake, the parameters and the caller's
 * slot array out_vertices [3][nsteps][m] (device, as streami_trace_streaklines) and allocates one
 * status byte per particle from the stream pool; _step advances k global steps (clamped to
 * nsteps; asynchronous); after s steps slot (j, i), j < s, holds the CURRENT position of particle
 * (i, j) (its last inside position if it died), identical to what streami_trace_streaklines would
 * return for nsteps = s; _position reports s; _end writes out_counts [m] (may be NULL) and
 * params->out_status, frees the handle and its scratch.  streami_trace_streaklines = begin,
 * step(nsteps), end.  All calls of one handle must use the same stream. */
typedef struct streami_streak_s* streami_streak;
int streami_streak_begin(streami_field f, const float* points, size_t m, unsigned nsteps,
                         const streami_params* params, float* out_vertices, void* cuda_stream,
                         streami_streak* out);
int streami_streak_step(streami_streak s, unsigned k, void* cuda_stream);
int streami_streak_position(streami_streak s, unsigned* steps_done /*host*/);
int streami_streak_end(streami_streak s, unsigned* out_counts, void* cuda_stream);

/* Polyline assembly (the paper's getLines / assembleOutput): one
 * contiguous AoS point buffer plus a per-line offset table, ready for a renderer or a writer.
 *   streami_streamline_lines: line id = the stored vertices of particle id in step order;
 *     vertices [3][n][capacity] and counts [n] as written by streami_trace_streamlines /
 *     streami_brick_advect.
 *   streami_streak_lines: line i = the particles of rake point i that are alive now, from the
 *     youngest release to the oldest, at the current step of the handle.
 * out_offsets [lines+1] device u64 (exclusive scan of the line lengths, last = total points);
 * out_points [total][3] device, or NULL to compute the offsets only (call once with NULL to learn
 * the total, allocate, call again); out_total HOST, may be NULL; when given the call synchronises
 * the stream. */
int streami_streamline_lines(const float* vertices, const unsigned* counts, size_t n, unsigned capacity,
                             unsigned long long* out_offsets, float* out_points,
                             unsigned long long* out_total, void* cuda_stream);
int streami_streak_lines(streami_streak s, unsigned long long* out_offsets, float* out_points,
                         unsigned long long* out_total, void* cuda_stream);

/* Streamlines end to end for a host application: seeds (host) in, assembled polylines (host) out
 * (f may be a monolithic or a bricked field: streami_trace_streamlines or streami_brick_advect runs):
 * out_offsets [n+1] u64 and out_points [max_points][3]; only the stored vertices cross the bus, not
 * the capacity-padded slot array.  params->capacity/stride select the vertices as usual; the
 * optional outputs in params are host pointers.  *out_total (host, may be NULL) = points of all
 * lines.  Large inputs run in up to 4 batches of seeds (option "host_batch"): the points of one batch
 * are copied out on a second, library-owned stream while the next batch is traced; pinned host
 * buffers are what lets that overlap happen, pageable ones work but serialise.  Synchronises
 * cuda_stream (once per batch: the batch's total sizes its device buffer) and returns with all copies
 * complete.  Returns STREAMI_E_TRUNCATED if total > max_points (the first max_points points are then
 * delivered). */
int streami_trace_streamlines_lines_host(streami_field f, const float* seeds, size_t n,
                                         const streami_params* params, unsigned long long* out_offsets,
                                         float* out_points, unsigned long long max_points,
                                         unsigned long long* out_total, void* cuda_stream);

/* streami_trace_streaklines / streami_brick_advect with HOST buffers (points/seeds, out_vertices,
 * out_counts, the optional outputs in params, the round table, the log and its count are host
 * pointers; pinned memory makes the copies faster but is not required): copy host->device, run,
 * copy device->host, synchronise cuda_stream before returning.  The round table keeps the caller's
 * content in the rows the call does not write. */
int streami_trace_streaklines_host(streami_field f, const float* points, size_t m, unsigned nsteps,
                                   const streami_params* params, float* out_vertices,
                                   unsigned* out_counts, void* cuda_stream);
int streami_brick_advect_host(streami_field f, const float* seeds, size_t n,
                              const streami_params* params, float* out_vertices, unsigned* out_counts,
                              unsigned* out_round_counts, unsigned max_rounds,
                              unsigned long long* out_handoff_log, size_t log_capacity,
                              unsigned long long* out_log_count, unsigned* out_nrounds,
                              void* cuda_stream);

/* Tuning knobs (process-wide).  None changes any result: they select schedules and staging only,
 * and exist so that each design choice can be measured A/B in one process.  name is one of
 *   "cell_cache"        0/1   keep the 8 cell vertices (streaklines: of both slices) in registers while samples stay in the cell
 *   "presort"           0/1   process work items in Morton order of their 4^3-cell block
 *   "segment_steps"     K     streamlines: K step attempts per particle per launch, survivors are
 *                             re-sorted between launches (0 = one launch; DP5(4) then synchronises)
 *   "prefetch"          0..4  RK4: request the cell the NEXT step is predicted to end in, a step ahead.  3 (default):
 *                             early form, issued right after stage 2 from p + 2 h k2; 4: also the next step's mid
 *                             point; 1: issued at the end of the step from p_new + (p_new - p) (2: plus the half-step
 *                             point); 0: off.  Bricked fields use the end-of-step form for every value > 0
 *   "integer_accept"    0/1   steady RK4 on a field of finite values: decide "inside" from floor(g)
 *   "vertex_staging"    0/1   stage vertices in shared memory and store full 32-byte sectors
 *   "max_blocks_per_sm" B     limit resident blocks per SM (0 = as many as fit)
 *   "brick_round_steps" k     brick rounds, see streami_brick_advect (-1, 0 = automatic, k > 0; -2 = one launch,
 *                             hand-offs through a device ring consumed by the same launch, if rounds are not observed)
 *   "streak_window"     W     streaklines: global steps per launch (0 = automatic)
 *   "host_batch"        S     streami_trace_streamlines_lines_host: seeds per batch (0 = automatic)
 *   "queue_steps"       Q     steady RK4 streamlines: a particle passes through a device queue, consumed by
 *                             the same launch, every Q steps, so that the launch runs breadth first and
 *                             ends without a long tail (0 = off, the default)
 *   "kernel_timing"     0/1   record a CUDA event pair around every advection-kernel launch
 * Returns INVALID for unknown names. */
int streami_set_option(const char* name, int value);
int streami_get_option(const char* name, int* value);


/* Number of kernels launched by this library since process start (for bench.py's gpu_launches). */
unsigned long long streami_launch_count(void);

/* With option "kernel_timing" = 1: device time (ms) of the advection-kernel launches recorded
 * since the previous call of this function, and how many there were; waits for those launches
 * to finish (event synchronise), then forgets them.  launches may be NULL. */
int streami_kernel_time(float* total_ms, unsigned* launches);

const char* streami_error_string(int code);

#ifdef __cplusplus
}
#endif
#endif /* STREAMI_H */
