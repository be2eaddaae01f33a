/*
 * haccsr.h -- C ABI of libhaccsr.so: HACC's short-range particle-particle force on one B200.
 *
 * What is computed (PAPER.md = arxiv 1410.2805; citations are PAPER.md lines):
 *
 *   "At distances less than the force-matching scale, r_s, the short-range force is given by
 *    subtracting the residual filtered grid force from the exact Newtonian force"
 *    (section 2.4), with the kernel of Eq. 12 (section 3.1)
 *
 *        f_SR(s) = (s + eps)^(-3/2) - f_grid(s),   s = r.r,
 *
 *    f_grid(s) "a 5-th order polynomial in s", eps the Plummer softening.  For every particle i
 *
 *        a_i = sum_{j != i, s_ij < r_max^2}  m_j * d_ij * f_SR(s_ij),
 *        d_ij = minimum image of (x_j - x_i) in the periodic box [0,L)^3,
 *
 *    found through a chaining mesh: particles binned into nc^3 cells of
 *    width L/nc >= r_max, each cell interacting with its 27 neighbours, followed
 *    by the kick map v <- v + dt*a.
 *
 * Conventions
 *   - Every pointer is a DEVICE pointer owned by the caller unless marked HOST.  The library
 *     never allocates or frees after haccsr_create and never frees caller memory.
 *   - Every call enqueues work on the CUDA stream given to haccsr_create and returns without
 *     synchronising (haccsr_sync / haccsr_get_stats synchronise).  Argument errors are returned
 *     synchronously; errors seen on the device (non-finite position) surface at haccsr_sync.
 *   - Return value: HACCSR_OK (0) or a negative haccsr_status.  No exceptions cross the ABI.
 *   - Particle arrays are float32 structure-of-arrays, lengths in grid units
 *     (PAPER.md:225), G = 1.
 *   - There is no CPU fallback: without a CUDA device every compute call returns HACCSR_ECUDA.
 */
#ifndef HACCSR_H
#define HACCSR_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct haccsr_ctx haccsr_ctx; /* opaque; owns no user memory */

typedef enum {
    HACCSR_OK = 0,
    HACCSR_EINVAL = -1, /* bad argument: nc < 4, L/nc < r_max, eps <= 0, n > n_max, NULL */
    HACCSR_ESTATE = -2, /* force before bin, kick before force                          */
    HACCSR_ENOMEM = -3, /* workspace too small                                          */
    HACCSR_ECUDA = -4,  /* CUDA runtime error (including: no device)                    */
    HACCSR_EDATA = -5   /* NaN/Inf position seen on the device                          */
} haccsr_status;

/* Version of this ABI (bumped when a signature changes). */
int haccsr_abi_version(void);

/* Bytes of device workspace haccsr_create needs for up to n_max particles on an nc^3 mesh.
 * Returns 0 for invalid arguments (n_max < 1, n_max >= 2^31, nc < 4, nc > 256). */
size_t haccsr_workspace_bytes(int64_t n_max, int nc);

/*
 * Create a context.  `workspace` (device, >= haccsr_workspace_bytes, 256-byte aligned) is
 * carved into the chaining mesh, the cell-ordered particle arrays and the work list -- the
 * "one preallocated pool" idea of PAPER.md:235.  box_L: periodic box length; nc: cells per
 * dimension (nc >= 4 so that the periodic image shift x - L is exact in float32 for the two
 * top cell layers and every periodic neighbour cell is distinct).  cuda_stream: a
 * cudaStream_t (NULL = default stream).  The context keeps the pointer; the caller keeps the
 * memory alive until haccsr_destroy.
 */
int haccsr_create(haccsr_ctx **out, int64_t n_max, float box_L, int nc, void *workspace,
                  size_t workspace_bytes, void *cuda_stream);
int haccsr_destroy(haccsr_ctx *ctx);

/*
 * Overloaded slab contexts -- HACC's particle overloading (section 2.2;
 * device blocks with r_s-wide boundary slabs PAPER.md:388-394, Fig. 13): "particles close to
 * the boundaries of their domain are replicated" in the neighbouring domain; the copies are
 * PASSIVE ("passive particles near the outer edge get no short-range force", they are
 * sources only) and the short-range step then needs no communication.
 *
 * A slab context covers the nz_own cell layers [cz_lo, cz_lo + nz_own) (mod nc) of the GLOBAL
 * nc^3 mesh of the periodic box, plus one passive layer below and one above (each L/nc >=
 * r_max wide).  1 <= nz_own <= nc - 2.  Positions stay in global box coordinates (no shift,
 * so every separation is computed from the same float32 numbers as in the whole box and
 * the interacting-pair set is identical); x and y are periodic, z neighbours come from the
 * window.  hacc_sr_bin on a slab context takes the owned particles AND the passive copies
 * (any order); a particle outside the window sets HACCSR_EDATA.  Particles in the two passive
 * layers get acceleration 0, neighbour count 0, and an unchanged velocity; pair_total and
 * the statistics count active targets only.  cell ids, cell_start and n_cells refer to the
 * window: id = cx + nc*(cy + nc*lz), lz = (cz - (cz_lo - 1)) mod nc in [0, nz_own + 2).
 */
size_t haccsr_workspace_bytes_slab(int64_t n_max, int nc, int nz_own);
int haccsr_create_slab(haccsr_ctx **out, int64_t n_max, float box_L, int nc, int cz_lo,
                       int nz_own, void *workspace, size_t workspace_bytes, void *cuda_stream);

/*
 * hacc_sr_pack_layer -- the message of the overloading exchange: append {x, y, z, m} (float4
 * records; positions wrapped into [0,L); m = 1 when mass is NULL) of every particle whose
 * position lies in GLOBAL cell layer cz_layer (cz = floor(z*nc/L) evaluated exactly) to
 * out_records[0 .. capacity).  *count (device uint32) receives the number of particles in
 * the layer; if it exceeds capacity only the first `capacity` slots were written and the
 * caller must retry with a larger buffer.  Order of the records is unspecified.
 * hacc_sr_unpack -- append n received records to SoA arrays (x, y, z, mass point at the first
 * free element; mass may be NULL).
 */
int hacc_sr_pack_layer(haccsr_ctx *ctx, int64_t n, const float *x, const float *y, const float *z,
                       const float *mass, int cz_layer, float *out_records, int64_t capacity,
                       uint32_t *count);
int hacc_sr_unpack(haccsr_ctx *ctx, int64_t n, const float *records, float *x, float *y, float *z,
                   float *mass);

/*
 * hacc_sr_bin -- build the chaining mesh (SoA + permutation array
 * PAPER.md:239, 307).
 *   cid_i = cx + nc*(cy + nc*cz), cx = floor(x_i*nc/L) evaluated exactly; the particles are
 *   counting-sorted by cell (three staged partition passes: z slab, y row, x cell) into
 *   cell-ordered float4 {x,y,z,m} with perm (sorted slot -> original index) and
 *   cell_start[nc^3+1] (exclusive prefix of the cell histogram); then the work list for the
 *   force kernel (dense cells split into target chunks x source chunks, PAPER.md:358 work queue).
 * x,y,z: length n, read only.  Positions outside [0,L) are wrapped (x - L*floor(x/L), a
 * result that rounds to L becomes 0); NaN/Inf sets HACCSR_EDATA.  mass: length n or NULL
 * (unit masses).  vx,vy,vz: length n or all NULL; they are remembered and updated in place by
 * hacc_sr_kick / hacc_sr_force_kick (original particle order; never permuted).
 * Within-cell order of the sorted arrays is unspecified (atomic ranks).
 */
int hacc_sr_bin(haccsr_ctx *ctx, int64_t n, const float *x, const float *y, const float *z,
                const float *mass, float *vx, float *vy, float *vz);

/*
 * hacc_sr_force -- short-range accelerations from the current mesh (Eq. 12).
 *   eps >= 1e-20 (units of s = length^2; the floor keeps eps^(-3/2) finite in float32 for
 *   the self pair and coincident pairs), 0 < r_max <= L/nc, poly: HOST pointer to c0..c5 of
 *   f_grid(s) = sum c_k s^k.  Cutoff is strict: a pair interacts iff s < r_max^2, decided on
 *   the exact value of s for the float32 inputs (FP32 fast path + FP64 recheck in a guard
 *   band), so neighbour counts are bit-exact.  j == i is excluded; coincident distinct
 *   particles count as a pair and contribute zero force.
 *   ax,ay,az: length n, ORIGINAL particle order, overwritten.
 *   nbr_count: length n (n_i = number of interacting neighbours) or NULL.
 *   pair_total: one uint64 (C = sum n_i, ordered pairs) or NULL.
 * The acceleration arrays are remembered for a following hacc_sr_kick.
 */
int hacc_sr_force(haccsr_ctx *ctx, float eps, float r_max, const float *poly /*HOST [6]*/,
                  float *ax, float *ay, float *az, uint32_t *nbr_count, uint64_t *pair_total);

/* hacc_sr_kick -- kick map: v <- v + dt * a(last hacc_sr_force), on the
 * velocity arrays given to hacc_sr_bin.  HACCSR_ESTATE if there is no force or no velocity. */
int hacc_sr_kick(haccsr_ctx *ctx, float dt);

/* Force with the kick fused into its epilogue: same result as hacc_sr_force followed by
 * hacc_sr_kick(dt) up to float32 rounding order (split dense cells add dt*a_partial). */
int hacc_sr_force_kick(haccsr_ctx *ctx, float eps, float r_max, const float *poly /*HOST*/,
                       float dt, float *ax, float *ay, float *az, uint32_t *nbr_count,
                       uint64_t *pair_total);

/* Stream map: x <- wrap(x + dt*v) into [0,L), in place, length n.
 * Independent of the mesh (call hacc_sr_bin again afterwards). */
int hacc_sr_drift(haccsr_ctx *ctx, int64_t n, float *x, float *y, float *z, const float *vx,
                  const float *vy, const float *vz, float dt);

/*
 * hacc_sr_subcycle -- the short-range map of Eq. 9: n_sub sub-cycles of the
 * symplectic "SKS" map (stream half a step, kick a full step with the force at
 * the streamed positions, stream half a step),
 *     M_sr(dt)^n_sub = S(dt/2) K(dt) [S(dt) K(dt)]^(n_sub-1) S(dt/2)
 * (adjacent half streams merged).  Every kick re-bins the streamed positions (hacc_sr_bin)
 * and evaluates the force (hacc_sr_force_kick); all of it is enqueued on the context's stream
 * without host synchronisation.  x,y,z,vx,vy,vz: length n, updated in place; mass: length n or
 * NULL; ax,ay,az: length n, receive the accelerations of the LAST kick.  n_sub >= 1 (the paper
 * uses 3-10).  Arguments as for hacc_sr_bin / hacc_sr_force; all of them are validated before
 * anything is enqueued, so an error return leaves x, y, z, v untouched.  On return the context holds the
 * mesh of the last kick's positions, which the final half stream has since moved.
 */
int hacc_sr_subcycle(haccsr_ctx *ctx, int64_t n, float *x, float *y, float *z, const float *mass,
                     float *vx, float *vy, float *vz, float eps, float r_max,
                     const float *poly /*HOST [6]*/, float dt, int n_sub, float *ax, float *ay,
                     float *az);

/*
 * hacc_sr_subcycle_multilevel -- one long step T of the short-range map with multi-level
 * (density-adaptive) time stepping, PAPER.md:214-216 (section 2.5) and 315-325 (section 3.1):
 * "particles in higher density regions will require finer short-range time steps", the density
 * estimate coming from the structure already built for the force -- here the occupancy n_c of
 * the particle's chaining-mesh cell at the BEGINNING of the long step.  Eq. 11:
 *     l = floor((rho/rho0) / d) + 1 kicks,  rho/rho0 = n_c * nc^3 / n,
 * raised to l_min and capped at l_max (both powers of two, l_max <= 64); a particle takes 2^k
 * kicks, k = floor(log2 l) its level (written to level[n], DEVICE uint8, original order).
 * Every particle is streamed by 2*l_max half streams of T/(2*l_max) ("all particles are acted
 * on by the same number of stream operators"); after half stream h the particles of level
 * k = log2(l_max) - (trailing zero bits of h) -- the midpoints of their 2^k SKS maps -- are
 * kicked by T/2^k with the force of ALL particles at the current positions: the mesh is
 * rebuilt with the particles of level k first in every cell, and they are the only targets
 * of the force evaluation (sources: everybody).  With l_min == l_max this is hacc_sr_subcycle with
 * n_sub = l_max, dt = T/l_max.  d > 0 is a float32 (the paper uses 10-20).
 * ax,ay,az receive the accelerations evaluated at the LAST kick (0 elsewhere).  evals (DEVICE
 * uint64, may be NULL) receives the candidate pairs evaluated over the whole step (the sum of
 * the n_eval statistics of its force evaluations).  Arguments are validated before anything
 * is enqueued; everything runs on the context's stream without host synchronisation.
 * Whole-box contexts only (HACCSR_EINVAL on a slab context: rho0 is the mean density of the
 * whole box, which a slab does not know).
 */
int hacc_sr_subcycle_multilevel(haccsr_ctx *ctx, int64_t n, float *x, float *y, float *z,
                                const float *mass, float *vx, float *vy, float *vz, float eps,
                                float r_max, const float *poly /*HOST [6]*/, float T, float d,
                                int l_min, int l_max, float *ax, float *ay, float *az,
                                uint8_t *level, uint64_t *evals);

/* Read-only views into context-owned device memory, valid until the next hacc_sr_bin.
 * Any out pointer may be NULL.  sorted_pos is float4 {x,y,z,m} per sorted slot. */
int haccsr_get_mesh(haccsr_ctx *ctx, const uint32_t **cell_start /*nc^3+1*/,
                    const uint32_t **perm /*n*/, const float **sorted_pos /*4n floats*/,
                    const uint32_t **cell_id /*n, original order*/);

typedef struct {
    int64_t n;                /* particles in the current mesh                              */
    int64_t n_cells;          /* nc^3                                                       */
    uint64_t n_eval;          /* sum_c n_c * sum_{27 nbrs} n_c' (candidate pairs incl. self) */
    uint32_t n_items;         /* work items the force kernel pulls                          */
    uint32_t n_split_items;   /* items whose source list was split (atomic combine)         */
    uint32_t max_cell_count;  /* largest cell occupancy                                     */
    uint32_t sources_per_split; /* source-chunk length used for splitting                  */
    uint64_t n_recheck_tiles; /* tiles that took the FP64 guard-band path in the last force */
} haccsr_stats;

/* Synchronises the stream and copies the statistics of the last bin/force to HOST. */
int haccsr_get_stats(haccsr_ctx *ctx, haccsr_stats *out /*HOST*/);

/* Stream synchronise + fetch (and clear) the device error flag. */
int haccsr_sync(haccsr_ctx *ctx);

const char *haccsr_strerror(int status);

/*
 * hacc_sr_cell_start_noalloc -- the chaining mesh's occupancy table without a context and
 * without ANY allocation (particles "sorted into" chaining-mesh cells; this is
 * the table of where each cell's particles start in that order).
 *
 * For callers that cannot call cudaMalloc or own a workspace (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid allocation).  Computes, for n particles at
 * x,y,z (DEVICE, float32[n], any real values: wrapped into [0,L) exactly as hacc_sr_bin wraps
 * them) on an nc^3 mesh over the periodic box of length box_L,
 *     cell_start[c] = number of particles in cells 0..c-1,  c = cx + nc*(cy + nc*cz),
 * for c = 0..nc^3 (cell_start[nc^3] = n): the same array haccsr_get_mesh returns after
 * hacc_sr_bin on a whole-box context.  cell_start: DEVICE, uint32[nc^3 + 1], caller-owned.
 *
 * Scratch (the per-cell counters) lives in a file-scope __device__ array of the library, of
 * HACCSR_NOALLOC_MAX_CELLS uint32 counters (1 MiB; every GPU that loads the library holds it
 * until the process exits).  Limit: nc <= 64, i.e.
 * nc^3 <= HACCSR_NOALLOC_MAX_CELLS; a larger mesh is refused with HACCSR_ENOMEM ("workspace
 * too small") and nothing is enqueued.  Other errors: HACCSR_EINVAL (nc < 4, n < 0, n >= 2^31,
 * box_L not positive and finite, a NULL pointer with n > 0, NULL cell_start), HACCSR_ECUDA.
 * Non-finite coordinates are counted in the cell of coordinate 0 (hacc_sr_bin's rule) and are
 * not reported.
 *
 * Runs on the device that is current at the call, on cuda_stream (a cudaStream_t of that
 * device, NULL = default stream); asynchronous.  Calls no cudaMalloc, cudaFree or allocating
 * library routine; the first call on a device looks the array's address up once
 * (cudaGetSymbolAddress), so make one warm-up call before a graph capture.  ALL calls in the
 * process share the one array per device: the call clears what it needs first, but two calls
 * that overlap on the GPU (different streams, no ordering between them) race and give wrong
 * tables.  Calls on one stream, or otherwise ordered, are safe.
 */
#define HACCSR_NOALLOC_MAX_NC 64
#define HACCSR_NOALLOC_MAX_CELLS (64 * 64 * 64)
int hacc_sr_cell_start_noalloc(int64_t n, const float *x, const float *y, const float *z,
                               float box_L, int nc, uint32_t *cell_start /*DEVICE*/,
                               void *cuda_stream);

/*
 * Peak probes behind the roofline denominator bench.py reports (not part of the method).
 * Each runs one register-only kernel on every SM and returns the elapsed milliseconds (CUDA
 * events on the given stream, best of `reps`) through *ms (HOST); *ops (HOST) receives the
 * operations executed.  kind 0: scalar FFMA (ops = FMAs), 1: packed fma.rn.f32x2 (ops = FMAs),
 * 2: MUFU rsqrt (ops = rsqrts).  No memory is allocated.  HACCSR_EINVAL for any other kind.
 */
int haccsr_probe_peak(int kind, int reps, void *cuda_stream, double *ms, double *ops);

#ifdef __cplusplus
}
#endif
#endif /* HACCSR_H */
