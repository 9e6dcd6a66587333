/*
 * srpp.h -- C ABI of the B200-native short-range particle-particle (PP) force solver.
 *
 * The hot path of HACC's short-range solver as the paper names it for accelerated systems
 * (PAPER.md = arXiv:1411.3396, Heitmann et al., "The Q Continuum Simulation"):
 *   PAPER.md:63 (Sec. 2)    force = long-range spectrally filtered PM + short-range solver; on
 *                           accelerated systems the short-range solver is a direct particle-particle
 *                           ("N^2") sum, i.e. "compute intensive".
 *   PAPER.md:65 (Sec. 2)    spectral filtering pushes the PM / short-range "hand-over" to small scales:
 *                           the pair force is Newtonian minus the filtered grid force, zero beyond rc.
 *   PAPER.md:73 (Sec. 2.1)  a "short-range force timestep" updates the particles (the kick).
 * PAPER.md prints no formula for this path; BASELINE.json `north_star` fixes its form and SURVEY.md 8(c)
 * lists the readings R1..R18 (repeated in DESIGN.md) that make it precise:
 *
 *   a_i = sum_{j, s_ij < rc^2}  m_j d_ij [ (s_ij + eps^2)^(-3/2) - P(s_ij) ],     s_ij = |d_ij|^2,
 *   d_ij = minimum image of x_j - x_i in the periodic box,  P(s) = sum_{k=0..5} poly[k] s^k,  G = 1.
 *
 * Conventions
 *   - Every array argument is a DEVICE pointer unless its name ends in `_host`.  float4 arrays are
 *     AoS (x, y, z, w), 16-byte aligned.  The caller owns all arrays and the workspace; the library
 *     owns only the small host-side context.  No call allocates device memory.
 *   - `cuda_stream` is a cudaStream_t passed as void* (0 = the legacy default stream).  Calls enqueue
 *     work on it and return; only srpp_build_mesh() synchronises the stream (it reads a device-side
 *     error flag), and the *_host convenience entry points synchronise because they copy.
 *   - Every call returns SRPP_OK (0) or a negative srpp_status; nothing throws or aborts across the ABI.
 *     There is no CPU fallback and no other back end: without a CUDA device every compute call
 *     returns SRPP_ERR_CUDA.
 *   - Units: PM grid units, G = 1, accelerations (no m_i factor).
 */
#ifndef SRPP_H_
#define SRPP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SRPP_VERSION 1

typedef enum {
  SRPP_OK = 0,
  SRPP_ERR_INVALID_ARG = -1, /* null or misaligned (16 B) pointer, n < 0 or n >= 2^31, eps <= 0, rcut <= 0,
                                non-finite parameter                                                         */
  SRPP_ERR_GEOMETRY = -2,    /* ncell < 3 on an axis, box/ncell < rcut, more than 2^24 cells (R8), or a box
                                length / cutoff above 2^24 grid units (fp32 exact-integer range)              */
  SRPP_ERR_DOMAIN = -3,      /* a position outside [0, L) or not finite, found while binning (R13)            */
  SRPP_ERR_WORKSPACE = -4,   /* workspace too small or not 256-byte aligned                                   */
  SRPP_ERR_STATE = -5,       /* srpp_accel before a successful srpp_build_mesh, n mismatch, or the current CUDA
                                device is not the one the context was created on                             */
  SRPP_ERR_CUDA = -6,        /* CUDA runtime error (text of the last one: srpp_last_cuda_error)                */
  SRPP_ERR_LIMIT = -7        /* a size beyond the fixed capacity of srpp_mbp_static's built-in scratch array     */
} srpp_status;

/* Solver parameters (plain data; copied by srpp_create). */
typedef struct {
  float box[3];      /* periodic box lengths Lx, Ly, Lz (> 0), grid units                                   */
  int32_t ncell[3];  /* chaining-mesh cells per axis (>= 3); cell edge = box/ncell must be >= rcut            */
  float rcut;        /* cutoff radius rc (> 0); a pair contributes iff s < rc^2, strictly (R5)                */
  float eps;         /* Plummer softening length (> 0); eps^2 is added to s in the Newtonian term only (R3)  */
  float poly[6];     /* c0..c5 of the grid-force fit P(s), s = r^2 (R4); see srpp_default_poly               */
} srpp_params;

typedef struct srpp_ctx srpp_ctx;

/* Counters of the last srpp_accel, for harness reporting (host memory). */
typedef struct {
  uint64_t work_items;      /* warp-level work items executed (target tile x source chunk)                  */
  uint64_t pair_slots;      /* pair evaluations issued, padding included                                     */
  uint64_t candidate_pairs; /* W = sum_c n_c * sum_{c' in 27-stencil(c)} n_c'             */
  uint32_t max_cell_count;  /* largest cell occupancy                                                       */
  uint32_t uniform_mass;    /* 1 if every particle carries the same mass (fast path taken)                   */
  uint64_t kernel_launches; /* CUDA kernels this context has launched since srpp_create (all calls)          */
  uint64_t rebins_incremental; /* re-bins inside srpp_subcycle done by the incremental merge ...               */
  uint64_t rebins_full;        /* ... and by a full rebuild (too many movers), since srpp_create                */
  uint64_t last_movers;        /* particles that changed cell in the last sub-step of the last srpp_subcycle    */
} srpp_stats;

/* Device times of the last srpp_build_mesh / srpp_accel, from CUDA events the library records on ITS
 * stream around each phase when timing is enabled (milliseconds; -1 where no phase has run yet). */
typedef struct {
  float mesh_ms;   /* A1-A4: all binning kernels of the last srpp_build_mesh                                */
  float accel_ms;  /* A5-A6: whole srpp_accel (work plan + PP force kernel + write-back)                     */
  float force_ms;  /* A5 only: the PP force kernel launch                                                    */
  float rebin_ms;  /* mean incremental re-bin of the last srpp_subcycle (movers' sort + merge)                */
  float kick_stream_ms; /* mean fused kick + stream + mover detection pass of the last srpp_subcycle          */
} srpp_timings;

/* The six default coefficients (degree-5 fit in s to a Gaussian-filtered point
 * mass, sigma = 1.2, with P(9) = 1/27), written to poly_host[6]. */
int32_t srpp_default_poly(float* poly_host);

/* Bytes of device workspace needed for n particles with these parameters (256-byte aligned base).
 * Holds: cell ids, radix-sort ping-pong keys/values and digit histograms, cell_start[ncells+1],
 * perm[n], sorted float4[n], per-cell work tables, fp64 accumulators double[3n], flags/counters. */
int32_t srpp_workspace_bytes(const srpp_params* params, int64_t n, size_t* bytes_host);

/* Validates `params`, records workspace + stream.  The context is host memory owned by the library. */
int32_t srpp_create(srpp_ctx** ctx, const srpp_params* params, void* workspace, size_t workspace_bytes,
                    void* cuda_stream);
void srpp_destroy(srpp_ctx* ctx);

/*
 * A1-A4: chaining mesh = stable counting sort of the particles by linear cell id.
 *   cell coordinate per axis in fp32: inv = (float)ncell/box; c = min((int)floorf(x*inv), ncell-1) (R10)
 *   cid = cx + ncx*(cy + ncy*cz) (R11); inside a cell, ascending original index (R12).
 * pos_mass: device float4[n] (x, y, z, m), read-only, 0 <= x < L required (else SRPP_ERR_DOMAIN).
 * Synchronises the stream once to read the error flag.  Results are bit-exact reproducible.
 */
int32_t srpp_build_mesh(srpp_ctx* ctx, const float* pos_mass, int64_t n);

/* Borrowed device views into the workspace, valid until the next srpp_build_mesh / srpp_destroy:
 *   cell_start uint32[ncells+1] (cell_start[ncells] = n), perm uint32[n] (perm[k] = original index of the
 *   k-th particle in (cid, index) order), sorted float4[n] (sorted[k] = pos_mass[perm[k]]).
 * Any of the three output pointers may be NULL. */
int32_t srpp_get_mesh(const srpp_ctx* ctx, const uint32_t** cell_start, const uint32_t** perm,
                      const float** sorted);

/* A5-A6: short-range accelerations of all n particles from the last mesh, written in the caller's
 * ORIGINAL particle order (R15) as float4 (ax, ay, az, 0).  fp32 pair arithmetic, MUFU rsqrt,
 * per-item fp32 partial sums folded into fp64 accumulators.  Asynchronous on the stream. */
int32_t srpp_accel(srpp_ctx* ctx, float* acc);

/* A5-A7 in one call: srpp_accel followed by srpp_kick(vel, acc, kdt) on the same n particles, with the kick fused into
 * the write-back (one pass over acc and vel instead of a scattered write of acc and a second pass that re-reads it).
 * Results are bit-identical to the two separate calls.  acc, vel: device float4[n], n = particles of the last mesh.
 * For n >= 2^22 the write-back is bucketed (two coalesced passes through a 16 n-byte buffer of the workspace) because
 * the destinations perm[k] have no locality.  Asynchronous on the stream.
 * Errors: INVALID_ARG (null / misaligned pointer, non-finite kdt), STATE, CUDA. */
int32_t srpp_accel_kick(srpp_ctx* ctx, float* acc, float* vel, float kdt);

/* Counters of the last srpp_accel (synchronises the stream). */
int32_t srpp_get_stats(srpp_ctx* ctx, srpp_stats* stats_host);

/* Enable (1) / disable (0) event recording around the phases; off by default.  srpp_get_timings
 * synchronises the stream and reads the events of the last build/accel. */
int32_t srpp_set_timing(srpp_ctx* ctx, int32_t enable);
int32_t srpp_get_timings(srpp_ctx* ctx, srpp_timings* timings_host);

/* FP32 peak probe for the "% of FP32 peak" report: runs a register-only FMA stream on
 * every SM of the context's device and writes the sustained flop/s to *flops_per_s_host.
 * variant 0 = scalar FFMA, 1 = packed FFMA2 (the pair loop's form), 2 / 3 = packed FFMA2 whose every
 * instruction reads 2 / 3 different vector registers (register-file operand bandwidth);
 * trips >= 1 scales the run time (trips = 2000 is about 10 ms).  Synchronises. */
int32_t srpp_probe_fp32(srpp_ctx* ctx, int32_t variant, int32_t trips, double* flops_per_s_host);

/* Overloaded (non-periodic) node volume and active/passive particles ("particle
 * overloading", PAPER.md:73 blocks of active and passive particles).  Optional; the default after srpp_create is a fully
 * periodic box in which every particle is active (BASELINE.json configs).
 *   periodic_host[3]   1 = periodic axis (minimum image), 0 = open axis: coordinate differences are taken as they are
 *                      and the 27-cell stencil stops at the box faces.  NULL = all periodic.
 *   active_lo_host[3], active_hi_host[3]   the active box.  Accelerations are computed for every particle in a
 *                      chaining-mesh cell that intersects [lo, hi) (a superset of the particles inside it); particles in
 *                      the other cells are passive: they act as sources only and their acceleration is written as 0.
 *                      NULL = the whole box.
 * Host pointers, read during the call.  Takes effect at the next srpp_accel (the mesh does not depend on it).
 * Errors: INVALID_ARG (null ctx, lo > hi, non-finite). */
int32_t srpp_set_boundary(srpp_ctx* ctx, const int32_t* periodic_host, const float* active_lo_host,
                          const float* active_hi_host);

/* Most-bound-particle halo centre finder ("identification of the halo center as
 * defined by its potential minimum (most bound particle)").  Reading R19: halo h is the contiguous run
 * pos_mass[halo_start[h] .. halo_start[h+1]) and, for every member i,
 *     phi_i = - sum_{j in h, j != i} m_j / sqrt(|x_j - x_i|^2 + eps^2)        (G = 1, eps of srpp_params, plain differences)
 * The centre is the member with the smallest phi (lowest index on ties).
 *   pos_mass          device float4[n]; positions need not lie in the box (no mesh is used)
 *   halo_start_host   HOST int64[nhalo+1], non-decreasing, within [0, n]; read (validated and uploaded) during the
 *                     call; nhalo <= 2^24
 *   phi               device float[n] or NULL: phi of every halo member (entries outside every halo are not written)
 *   mbp_index         device int64[nhalo]: index into pos_mass of each halo's centre, -1 for an empty halo
 *   mbp_phi           device float[nhalo] or NULL: its potential (0 for an empty halo)
 *   workspace         device, 256-byte aligned, >= srpp_mbp_workspace_bytes(n, nhalo); owned by the caller
 * Pair arithmetic in fp32 (partial sums of <= 1024 terms folded in fp64; the argmin is taken on those fp64 sums).
 * Asynchronous on the context's stream: the item prefix is computed on the device, no synchronisation.
 * Errors: INVALID_ARG, WORKSPACE, STATE (another device is current), CUDA. */
int32_t srpp_mbp_workspace_bytes(int64_t n, int64_t nhalo, size_t* bytes_host);
int32_t srpp_mbp(srpp_ctx* ctx, const float* pos_mass, int64_t n, const int64_t* halo_start_host, int64_t nhalo,
                 float* phi, int64_t* mbp_index, float* mbp_phi, void* workspace, size_t workspace_bytes);

/* srpp_mbp for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the same computation as srpp_mbp -- same kernels, same reading R19, same outputs --
 * but with NO workspace argument and no context.  The scratch memory (fp64 potential accumulators, the halo table, the work-item
 * prefix, the queue counter) lives in one static __device__ array inside the library, sized for
 *     n <= SRPP_MBP_STATIC_MAX_N (2^20 members)  and  nhalo <= SRPP_MBP_STATIC_MAX_HALOS (2^16 halos),
 * about 9.1 MB, which every GPU that loads the library holds until the process exits.  A larger n or nhalo is rejected with
 * SRPP_ERR_LIMIT (use srpp_mbp with a caller-owned workspace instead).  The call allocates nothing: no cudaMalloc, no cudaFree,
 * no allocating library routine; it only enqueues memsets, one copy of the halo table and the kernels on `cuda_stream`.
 *   pos_mass, phi, mbp_index, mbp_phi, halo_start_host   as for srpp_mbp (phi and mbp_phi may be NULL)
 *   eps               Plummer softening length (> 0, finite); srpp_mbp takes it from its context
 *   cuda_stream       cudaStream_t as void* (0 = the legacy default stream); asynchronous, no synchronisation
 * The array is SHARED by every call on a device and keeps the last call's contents; each call clears the parts that must
 * start at zero (queue counter, accumulators of the n members it uses).  Two calls whose GPU work overlaps (different
 * streams, or host threads that do not order their calls) RACE on it: order them on one stream or with events.
 * The first call on each device looks the array's device address up (cudaGetSymbolAddress, with that device current) and
 * queries the SM count and the kernel's occupancy; make that first call outside a stream capture.
 * Errors: INVALID_ARG (null / misaligned pointer, n or nhalo < 0, eps <= 0 or non-finite, halo table not monotone or beyond n),
 * LIMIT (n or nhalo above the maxima), STATE (device index above 63), CUDA. */
#define SRPP_MBP_STATIC_MAX_N (1 << 20)
#define SRPP_MBP_STATIC_MAX_HALOS (1 << 16)
int32_t srpp_mbp_static(const float* pos_mass, int64_t n, const int64_t* halo_start_host, int64_t nhalo, float eps,
                        float* phi, int64_t* mbp_index, float* mbp_phi, void* cuda_stream);

/* Block decomposition of the node volume with the x2 adaptive refinement rule (PAPER.md:73-77:
 * "1) Each node partitions itself into overlapping data blocks, 2) evolves the blocks independently, and 3) reconciles the
 * alive particles, whereby removing the unnecessary duplicated passive ones"; "the x-axis is equally partitioned in PM
 * grid units"; a block whose "timing is more than a factor of two larger than the average" is "divided a factor of two
 * finer").  One GPU evaluates the blocks one after the other; each block is an independent problem: its particles (the
 * active x-range plus a passive shell of >= rcut on both sides, through the periodic face if x is periodic) are extracted
 * into their own arrays in a block-local frame, get their own chaining mesh with OPEN x faces and their own force
 * evaluation, and only the active particles' accelerations are written back.
 *   srpp_blocks_init      (re)starts the plan with nblocks equal x-ranges, boundaries at integer grid units (box[0] must be
 *                         integer-valued and >= nblocks, else GEOMETRY; 1 <= nblocks <= SRPP_MAX_BLOCKS)
 *   srpp_accel_blocks     accelerations of all n particles (caller's order, .w = 0), block by block, from the positions
 *                         given here (the context's own mesh is neither used nor changed).  Every block is timed on the
 *                         device; afterwards the plan for the NEXT call is refined by the x2 rule.  The y/z periodic flags
 *                         of srpp_set_boundary apply; its active box does not.  Synchronises per block.
 *                         workspace: device, 256-byte aligned, >= srpp_blocks_workspace_bytes(params, n).
 *   srpp_get_blocks       the blocks of the last srpp_accel_blocks (host array), with their device times.
 * Block-local coordinates are exact in fp32 (integer frame origins) except for the shell that wraps through the face
 * x = box[0]; results agree with the periodic evaluation within the north_star tolerances (tested).
 * Errors: INVALID_ARG, GEOMETRY, WORKSPACE, STATE (no plan / other device), DOMAIN, CUDA. */
#define SRPP_MAX_BLOCKS 64
typedef struct {
  float x0, x1;              /* active range [x0, x1), grid units                                                  */
  int32_t level;             /* refinement level (0 = initial partition)                                           */
  int32_t pad_;
  int64_t n_active, n_total; /* active particles / particles incl. the passive shell                               */
  uint64_t candidate_pairs;  /* W of the block's own mesh (sum over blocks / W of the box = duplicated work)        */
  float ms;                  /* device time of the block: extract + mesh + force + reconcile                       */
  float pad2_;
} srpp_block_info;
int32_t srpp_blocks_workspace_bytes(const srpp_params* params, int64_t n, size_t* bytes_host);
int32_t srpp_blocks_init(srpp_ctx* ctx, int32_t nblocks);
int32_t srpp_accel_blocks(srpp_ctx* ctx, const float* pos_mass, int64_t n, float* acc, void* workspace,
                          size_t workspace_bytes);
int32_t srpp_get_blocks(const srpp_ctx* ctx, srpp_block_info* blocks_host, int32_t capacity, int32_t* count_host);

/* A7: sub-cycled kick, v <- fmaf(a, kdt, v) per component in fp32 (R16); .w lanes untouched.
 * vel, acc: device float4[n].  Asynchronous. */
int32_t srpp_kick(srpp_ctx* ctx, float* vel, const float* acc, float kdt, int64_t n);

/* Stream (drift): x <- wrap(fmaf(v, dt, x)) per component in fp32, result in [0, L) (a value that rounds
 * to L becomes 0; R13, R17).  Requires |v*dt| < L.  pos_mass is updated in place.  Asynchronous. */
int32_t srpp_stream(srpp_ctx* ctx, float* pos_mass, const float* vel, float dt, int64_t n);

/* The short-range sub-cycle as one call ("short-range force timestep": evolve, update the active
 * particles, stream the passive ones; reading R20 in DESIGN.md): nsub times
 *     x <- stream(x, v, dt/2);   a = accel(x);   v <- kick(v, a, kdt);   x <- stream(x, v, dt/2)
 * with srpp_stream / srpp_build_mesh + srpp_accel / srpp_kick semantics for the three pieces (dt/2 = the fp32 product
 * 0.5f*dt; with an active box set by srpp_set_boundary the passive particles have a = 0 and are only streamed).
 *   pos_mass, vel   device float4[n], updated in place
 *   acc             device float4[n]: accelerations of the LAST sub-step, caller's order (.w = 0)
 * On return the chaining mesh held by the context is the mesh of the RETURNED positions (srpp_get_mesh, or a following
 * srpp_accel, may use it).  Between the first and the last sub-step the state stays in chaining-mesh order: kick and
 * streams are one coalesced pass over the force kernel's accumulators, and the mesh is repaired by an incremental
 * re-bin (only the particles that changed cell are sorted and merged back; result bit-identical to a full build), with
 * a full rebuild as fall-back when more than n/4 particles changed cell.  Synchronises the stream once per sub-step.
 * Errors: INVALID_ARG (null / misaligned pointer, nsub < 0, non-finite dt or kdt), WORKSPACE, DOMAIN, STATE, CUDA. */
int32_t srpp_subcycle(srpp_ctx* ctx, float* pos_mass, float* vel, float* acc, float dt, float kdt, int32_t nsub,
                      int64_t n);

/* End-to-end convenience for callers holding HOST arrays: copies pos_mass_host[4n] (and vel_host[4n] if
 * not NULL) to the device, builds the mesh, computes accelerations, optionally kicks (vel_host != NULL:
 * v <- v + kdt*a, copied back), copies acc back to acc_host[4n].  Device scratch for the particle arrays
 * is taken from `device_scratch` (>= 48*n bytes, caller-owned device memory).  The velocity upload and the download
 * of the accelerations run on a second stream and overlap the kernels (host buffers should be pinned).  Synchronises. */
int32_t srpp_step_host(srpp_ctx* ctx, const float* pos_mass_host, float* vel_host, float* acc_host,
                       float kdt, int64_t n, void* device_scratch, size_t device_scratch_bytes);

/* Static strings. */
const char* srpp_strerror(int32_t status);
const char* srpp_last_cuda_error(const srpp_ctx* ctx);
int32_t srpp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SRPP_H_ */
