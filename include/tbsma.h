/*
 * tbsma.h -- C ABI of libtbsma: batched TB-SMA (Au) force evaluation + MD step on one B200.
 *
 * The method is the second-moment tight-binding potential of arXiv:1311.3890, section 2.1
 * ("P:NN" = line NN of /root/reference/PAPER.md; "D:Ak" = reading Ak in DESIGN.md):
 *     rho_i = sum_j xi^2 exp(-2q (r_ij/r0 - 1))                       P:47 Eq.1
 *     E_i   = sum_j A exp(-p (r_ij/r0 - 1)) - sqrt(rho_i)              P:47-55 Eq.1-3
 *     F_i   = -dE_C/dr_i, which needs rho_i and rho_j
 * evaluated "in two stages (two CUDA kernels), each stage looping over atom i's neighbors"
 * over a cutoff neighbour list with a buffer radius, inside a velocity-Verlet
 * step of 2 fs with rigid gripping layers.  Many independent nanowire replicas are
 * processed by every launch (the paper's science is > 2000 independent runs).
 *
 * Conventions
 *   - Units: Angstrom, eV, fs, amu, K.  1 eV/(A amu) = 9.648533212e-3 A/fs^2,
 *     kB = 8.617333262e-5 eV/K.
 *   - "d_" pointers are DEVICE memory owned by the caller; "h_" pointers are HOST memory.
 *     The context owns only its scratch (cells, lists, positions at build time, 1/sqrt(rho)).
 *   - pos / vel / force_energy are arrays of n_atoms x 4 floats (float4, 16-byte aligned):
 *       pos   = (x, y, z, flag)   flag = int32 bit pattern: 0 dynamic, 1 fixed grip, 2 pulled grip
 *       vel   = (vx, vy, vz, zref) zref = reference z of a grip atom; a pulled atom is PLACED at
 *                                  zref + D_r every step (D:A10, fp64 displacement, never
 *                                  incremented in fp32); ignored for dynamic atoms
 *       force_energy = (Fx, Fy, Fz, E_i)
 *   - Atoms of replica r occupy the index range [off[r], off[r+1]) at all times.  Inside that
 *     range tbsma_build_cells permutes atoms into cell order IN PLACE and records the original
 *     index of every slot in d_tag; everything the caller compares is compared in tag space.
 *   - Every call is asynchronous on `stream` (a cudaStream_t passed as void*; NULL = default
 *     stream) and never synchronises, except tbsma_status, tbsma_count_pairs, tbsma_get_stats
 *     and the *_host entry point.  Calls are safe to capture into a CUDA graph.
 *   - Errors: every function returns TBSMA_OK (0) or a negative code; nothing throws or aborts.
 *     Asynchronous faults (list overflow, skin violated, ...) are reported by tbsma_status.
 *   - There is no CPU fallback: without a CUDA device every call returns TBSMA_ECUDA.
 */
#ifndef TBSMA_H
#define TBSMA_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tbsma_ctx tbsma_ctx; /* opaque */

/* Table 1 of the paper; r0 is the first-neighbour distance a/sqrt(2) (D:A1). */
typedef struct {
    double A, xi, p, q, r0, mass_amu;
} tbsma_params;

enum {
    TBSMA_OK = 0,
    TBSMA_EINVAL = -1, /* bad argument (NULL, negative size, box shorter than 2 (r_cut+skin) on a periodic axis) */
    TBSMA_ENOMEM = -2, /* device or host allocation failed */
    TBSMA_ECUDA = -3,  /* a CUDA runtime call failed (or no device) */
    TBSMA_ESTATE = -4, /* call order violated (e.g. compute before build_neighbors) */
    TBSMA_ELIMIT = -5  /* a size exceeds the fixed capacity of a no-allocation entry point (tbsma_kinetic_tensor_noalloc) */
};

/* bits of the status word returned by tbsma_status */
enum {
    TBSMA_FLAG_NLIST_OVERFLOW = 1u, /* an atom had more than max_neighbors partners: list truncated, results invalid */
    TBSMA_FLAG_OUT_OF_BOX = 2u,     /* an atom left its replica's (non-periodic) box: still correct, edge cells grow */
    TBSMA_FLAG_NONFINITE = 4u,      /* a non-finite force was produced */
    TBSMA_FLAG_SKIN_VIOLATED = 8u,  /* with a fixed rebuild cadence an atom moved more than skin/2 between rebuilds */
    TBSMA_FLAG_TILE_OVERFLOW = 16u  /* shared-memory variant: a tile's halo outgrew its shared-memory image (sized at
                                       tbsma_build_cells from the populations found then, with 25 % headroom for layer
                                       tiles and 2.5 - 10 % for box tiles, as much as costs no residency); that tile was
                                       skipped, results invalid: call tbsma_build_cells again, or use variant 1 */
};

typedef struct {
    uint64_t n_steps;          /* md steps taken since tbsma_set_system */
    uint64_t n_replica_builds; /* neighbour-list builds, counted per replica (both kinds, see tbsma_set_outer_skin) */
    uint64_t n_build_passes;   /* steps (or explicit calls) in which at least one replica was rebuilt */
    int32_t max_neighbors_seen;
    int32_t n_candidate_builds; /* of those, builds that also redid the cells and the candidate list (saturating) */
} tbsma_stats;

/* Create a context for one parameter set.  r_cut: interaction cutoff, plain truncation, strict
 * r < r_cut (D:A4).  skin: neighbour-list buffer radius r_buff. */
int tbsma_create(const tbsma_params *params, double r_cut, double skin, tbsma_ctx **out);
int tbsma_destroy(tbsma_ctx *ctx);

/* Describe the batch: n_replicas independent systems, atoms of replica r are
 * [h_replica_offsets[r], h_replica_offsets[r+1]).  h_box_lo / h_box_hi: n_replicas x 3 floats;
 * h_periodic: n_replicas x 3 bytes (wires: 0,0,0; bulk: 1,1,1; D:A7).  On a periodic axis the box
 * length is the fp32 difference hi - lo and must be >= 2 (r_cut + skin); positions must lie in
 * [lo, hi).  On a non-periodic axis the box only sizes the cell grid (size it for the longest
 * elongation expected; atoms outside are binned into the edge cells and flagged OUT_OF_BOX).
 * max_neighbors: list capacity per atom (rounded up to a multiple of 4).  The perfect fcc lattice has 86 partners
 * within r_cut + skin = 7.3 A; a 3 nm wire at 298 K under tension reached 97 in 5000 steps, so 112 is the binding's default.
 * All arguments are HOST pointers; (re)allocates the context's device scratch. */
int tbsma_set_system(tbsma_ctx *ctx, int64_t n_atoms, int32_t n_replicas,
                     const int32_t *h_replica_offsets, const float *h_box_lo,
                     const float *h_box_hi, const uint8_t *h_periodic, int32_t max_neighbors);

/* Cell binning (counting sort over replica x cell keys, stable by tag inside a cell) and in-place
 * reorder of d_pos, d_vel (nullable) and d_tag into cell order; positions on periodic axes are
 * wrapped into [lo, hi).  d_tag must hold the current tag of every slot (0..n-1 before the
 * first call).  Rebuilds every replica.  The caller's force array is NOT permuted: after this call (and
 * tbsma_build_neighbors) evaluate tbsma_compute before the next tbsma_md_step / tbsma_md_run. */
int tbsma_build_cells(tbsma_ctx *ctx, float *d_pos, float *d_vel, int32_t *d_tag, void *stream);

/* Neighbour list of every atom: all j != i of the same replica with |r_i - r_j| < r_cut + skin,
 * membership decided by the fp32 predicate of D:A6.  Must directly follow tbsma_build_cells on the
 * same d_pos / d_vel (nullable) / d_tag.  The shared-memory variant additionally reorders the atoms
 * inside every z-layer of cells by neighbour count (longest lists first, ties by slot) and permutes
 * d_pos, d_vel and d_tag accordingly; the global variant leaves them untouched. */
int tbsma_build_neighbors(tbsma_ctx *ctx, float *d_pos, float *d_vel, int32_t *d_tag, void *stream);

/* One force evaluation (stage 1 densities, stage 2 forces) over the current list.
 * d_force_energy: out, n x 4 (F_i, E_i).  d_replica_energy: out, n_replicas doubles, E_C of each
 * replica (Eq.3).  d_replica_virial: out or NULL, n_replicas x 6 doubles, W_ab = 1/2 sum_i sum_j
 * d_ij,a f_ij,b in the order xx yy zz xy xz yz (potential part of Eq.5; D:A11). */
int tbsma_compute(tbsma_ctx *ctx, const float *d_pos, float *d_force_energy,
                  double *d_replica_energy, double *d_replica_virial, void *stream);
/* (Shared-memory variant: the per-replica sums of tbsma_compute / tbsma_md_step / tbsma_md_run are added in a fixed
 * order -- the 32 atoms of a chunk by a shuffle tree, the chunks of a CTA in chunk order, the CTAs of a replica in tile
 * order -- and are bitwise repeatable from run to run; the global variant adds them with fp64 atomics.) */

/* One MD step of every replica (thermostat D:A8 = BAOAB Langevin, gamma = 0 is exactly
 * velocity Verlet):  B A O A, neighbour rebuild of the replicas whose atoms moved more than
 * skin/2 since their last build (D:A14), forces, B.  On entry d_force_energy must hold the
 * forces of d_pos (from tbsma_compute or the previous step); on exit pos, vel, force are those
 * of the next step.  d_T: n_replicas floats (K); gamma_per_fs: friction; d_seed: n_replicas
 * uint64 Philox keys; step: the counter that, with the atom's tag inside its replica, selects
 * the noise (D:A9); d_slab_disp: n_replicas doubles, TOTAL displacement D_r of the pulled slab
 * (NULL = 0).  Outputs d_replica_energy / d_replica_virial / d_replica_ekin (eV, dynamic atoms,
 * after the final B) may each be NULL.  d_vel and d_tag are permuted with d_pos on rebuilds. */
int tbsma_md_step(tbsma_ctx *ctx, float *d_pos, float *d_vel, float *d_force_energy,
                  int32_t *d_tag, double dt_fs, const float *d_T, double gamma_per_fs,
                  const uint64_t *d_seed, uint64_t step, const double *d_slab_disp,
                  double *d_replica_energy, double *d_replica_virial, double *d_replica_ekin,
                  void *stream);

/* n_steps MD steps, steps step0 .. step0+n_steps-1, the pulled slab of replica r at
 * D_r(s) = d_slab_disp0[r] + d_slab_rate[r] * (s + 1 - step0) during step s (both nullable = 0).
 * rebuild_every > 0 additionally rebuilds every replica whenever s % rebuild_every == 0 and
 * raises SKIN_VIOLATED if an atom nevertheless moved more than skin/2 (BASELINE config 5).
 * The per-replica outputs are those of the last step.  One launch set per step for all replicas;
 * no host synchronisation. */
int tbsma_md_run(tbsma_ctx *ctx, float *d_pos, float *d_vel, float *d_force_energy,
                 int32_t *d_tag, double dt_fs, const float *d_T, double gamma_per_fs,
                 const uint64_t *d_seed, uint64_t step0, int64_t n_steps,
                 const double *d_slab_disp0, const double *d_slab_rate, int32_t rebuild_every,
                 double *d_replica_energy, double *d_replica_virial, double *d_replica_ekin,
                 void *stream);

/* Same as tbsma_md_run but with HOST buffers: copies pos, vel, tag, T, seed, slab arrays to
 * the device, builds cells + lists, evaluates the initial forces, runs n_steps, and copies pos,
 * vel, force_energy, tag and the per-replica outputs back.  Synchronises.  h_tag in/out. */
int tbsma_md_run_host(tbsma_ctx *ctx, float *h_pos, float *h_vel, float *h_force_energy,
                      int32_t *h_tag, double dt_fs, const float *h_T, double gamma_per_fs,
                      const uint64_t *h_seed, uint64_t step0, int64_t n_steps,
                      const double *h_slab_disp0, const double *h_slab_rate, int32_t rebuild_every,
                      double *h_replica_energy, double *h_replica_virial, double *h_replica_ekin);

/* Observables of the tensile tests.  Eq.5 is garbled in the source (D:A11); it stands for the virial
 * stress  sigma_ab = -(W_ab + K_ab) / V,  tension positive, with W_ab the virial tbsma_compute / tbsma_md_step return,
 * K_ab = sum_i m v_a v_b over the dynamic atoms, and V the constant "hard-sphere" volume of the wire, which is the
 * caller's: tbsma_kinetic_tensor writes K of every replica (n_replicas x 6 doubles, eV, xx yy zz xy xz yz) for the
 * velocities in d_vel (flags from d_pos); tbsma_stress combines them (d_k may be NULL = 0 K) with d_volume
 * (n_replicas doubles, A^3) into d_sigma (n_replicas x 6, eV/A^3; 1 eV/A^3 = 160.21766208 GPa).  Strain (Eq.4)
 * is (L - L0) / L0 with L - L0 the slab displacement the caller itself supplies to tbsma_md_step. */
int tbsma_kinetic_tensor(tbsma_ctx *ctx, const float *d_pos, const float *d_vel, double *d_replica_kinetic, void *stream);
int tbsma_stress(tbsma_ctx *ctx, const double *d_replica_virial, const double *d_replica_kinetic,
                 const double *d_volume, double *d_sigma, void *stream);

/* tbsma_kinetic_tensor for callers that cannot allocate device memory.
 *
 * Everything else in this header needs a tbsma_ctx, and a context gets its tables from cudaMalloc (tbsma_set_system,
 * tbsma_build_cells).  That rules the library out for a caller whose process has already handed the GPU's memory to a pool
 * of its own (an MD engine or a training framework this code is plugged into: a cudaMalloc there fails, or takes memory the
 * pool's owner counts as its own), for a hook that runs between the steps of a loop that must not stall (cudaMalloc and
 * cudaFree synchronise the whole device), and for a job that was given a fixed memory budget.  This one call needs no
 * context and calls no cudaMalloc, cudaFree or other allocating routine, on its first call or any later one.
 *
 * It computes what tbsma_kinetic_tensor computes, K_ab = sum_i m v_i,a v_i,b over the dynamic atoms (flag 0 in pos.w) of
 * every replica, in eV, order xx yy zz xy xz yz (Eq.5 as read in D:A11), from
 *   d_pos, d_vel          n_atoms x 4 floats each, DEVICE, the layouts of the top of this file (only pos.w and vel.xyz
 *                         are read)
 *   d_replica_offsets     n_replicas + 1 int32, DEVICE (not host, unlike tbsma_set_system): atoms of replica r are
 *                         [off[r], off[r+1]); an empty replica gets K = 0
 *   mass_amu              atomic mass (tbsma_params.mass_amu)
 *   d_replica_kinetic     out, n_replicas x 6 doubles, DEVICE; overwritten, need not be cleared
 * asynchronously on `stream`.  All buffers stay the caller's.  The sums are added in a fixed order (which depends on
 * n_atoms, n_replicas and the offsets only), so the result is bitwise repeatable; it agrees with tbsma_kinetic_tensor,
 * which adds with atomics, to fp64 rounding.
 *
 * The working memory of the kernel (per-slice partial sums and one counter per replica) is a fixed array of
 * TBSMA_NOALLOC_SCRATCH_BYTES (784 KiB) inside the library's device code.  Consequences a caller must know:
 *   - Limits: n_replicas <= TBSMA_NOALLOC_MAX_REPLICAS (4096) and n_atoms <= TBSMA_NOALLOC_MAX_ATOMS (int32 offsets).
 *     Beyond them the call does nothing and returns TBSMA_ELIMIT; split the batch into several calls.
 *   - Every GPU on which the CUDA runtime loads this library holds those 784 KiB until the process exits, used or not.
 *   - There is one array per GPU, shared by all callers, threads and streams of the process.  Calls that can execute on
 *     the same GPU at the same time (different streams with no dependency between them) overwrite each other's partial
 *     sums and counters: wrong results, no error.  Put the calls on one stream or order them with events.  Calls that run
 *     one after the other need no care: the array keeps the previous call's contents, and every call first clears the
 *     counters it will use (on `stream`) and writes every partial sum before reading it.
 *   - The first call on a GPU (with that GPU current) looks up the array's device address and caches it; the runtime may
 *     load the library's device code at that point.  Make that first call before you begin any stream capture.
 * Errors: TBSMA_EINVAL (NULL pointer, negative size, mass <= 0), TBSMA_ELIMIT, TBSMA_ECUDA (no device, launch failed). */
#define TBSMA_NOALLOC_MAX_REPLICAS 4096
#define TBSMA_NOALLOC_MAX_SLOTS 16384 /* (replica, slice) partial sums; slices per replica = min(256, 16384 / n_replicas, ...) */
#define TBSMA_NOALLOC_MAX_ATOMS 2147483647
#define TBSMA_NOALLOC_SCRATCH_BYTES 802816 /* 4096 x 4 + 16384 x 6 x 8 */
int tbsma_kinetic_tensor_noalloc(const float *d_pos, const float *d_vel, const int32_t *d_replica_offsets,
                                 int64_t n_atoms, int32_t n_replicas, double mass_amu, double *d_replica_kinetic,
                                 void *stream);

/* Neighbour lists in TAG space for parity checks: d_counts[t] and d_list[t*max_neighbors + k]
 * (k < count, unsorted) for the atom whose tag is t.  d_tag as left by tbsma_build_cells. */
int tbsma_get_neighbors(tbsma_ctx *ctx, const int32_t *d_tag, int32_t *d_counts, int32_t *d_list,
                        void *stream);

/* Number of directed (i,j) list entries and of directed in-cutoff pairs for d_pos (synchronises). */
int tbsma_count_pairs(tbsma_ctx *ctx, const float *d_pos, int64_t *h_list_entries,
                      int64_t *h_cutoff_pairs, void *stream);

int tbsma_status(tbsma_ctx *ctx, uint32_t *h_flags); /* synchronises the device; clears nothing */
int tbsma_clear_status(tbsma_ctx *ctx);
int tbsma_get_stats(tbsma_ctx *ctx, tbsma_stats *h_out); /* synchronises */

/* Selects the neighbour-gather kernel variant (takes effect at the next tbsma_build_cells):
 *   1 = thread per atom over a k-major int32 list, neighbour records gathered from global memory
 *       through L1 (any system, periodic or not);
 *   2 = shared-memory tiles: a CTA stages the positions of a tile of cells (a run of z-layers of a thin wire, a box of
 *       cells of a thick wire or of a periodic replica) and of the cells around it in shared memory; 16-bit list
 *       entries, atoms ordered by list length inside a layer (or cell), lists ordered for conflict-free shared-memory
 *       gathers.  tbsma_build_cells returns TBSMA_EINVAL if a replica does not fit (a periodic axis shorter than three
 *       cells of r_cut + skin + S, a cell neighbourhood of more than 4095 atoms);
 *   0 = auto (default): 2 when it fits, else 1.
 * tbsma_get_variant returns the variant the current lists were built for. */
int tbsma_set_variant(tbsma_ctx *ctx, int32_t variant);
int tbsma_get_variant(const tbsma_ctx *ctx);
/* What the current lists were built for (each pointer may be NULL): number of tiles (0 under the global variant), whether
 * some replica is cut into boxes of cells rather than layers (tbsma_set_tile_box), whether the gather passes run as
 * persistent kernels (tbsma_set_gather). */
int tbsma_get_tiling(const tbsma_ctx *ctx, int32_t *n_tiles, int32_t *box_tiles, int32_t *persistent);

/* Shared-memory variant: buffer radius S of the CANDIDATE list (default 2.5 A).  The cell scan collects every
 * pair within r_cut + skin + S, once; while no atom has moved more than S/2 since then, the replica's list
 * (radius r_cut + skin) is re-filtered from those candidates whenever its atoms have moved more than skin/2
 * (inside the density pass of that step).  Membership of the list is decided by the predicate of D:A6 either way,
 * so S changes cost, never results; SKIN_VIOLATED is raised if candidates were used beyond their validity.
 * Takes effect at the next tbsma_build_cells. */
int tbsma_set_outer_skin(tbsma_ctx *ctx, double outer_skin);

/* Shape of the shared-memory tiles: own z-layers of cells per tile (1..8, default 2; a replica whose
 * layers are too populated gets fewer) and threads per CTA of the two gather kernels (multiple of
 * 32, <= 512, default 256).  Takes effect at the next tbsma_build_cells. */
int tbsma_set_tile(tbsma_ctx *ctx, int32_t layers_per_tile, int32_t threads);

/* Shared-memory variant: CTAs of the two gather kernels per tile.  0 (default) = automatic: one, unless the batch has
 * too few tiles to fill the GPU (a single 3 nm x 6 nm wire is 3 tiles), in which case several CTAs share a tile -- each
 * stages the tile image and takes a share of its 32-atom chunks -- until there are about eight CTAs per SM or one chunk
 * per CTA.  Changes cost and the order of the per-replica sums, nothing else.  Takes effect at the next
 * tbsma_build_cells. */
int tbsma_set_tile_split(tbsma_ctx *ctx, int32_t ctas_per_tile);

/* Shared-memory variant: a replica whose z-layers of cells fit a tile image (the paper's thin wires) is cut into runs of
 * whole layers; thicker wires and periodic replicas are cut into boxes of up to 3 x 3 x 3 cells with a one-cell halo,
 * wrapped around on periodic axes.  force != 0 cuts EVERY replica into boxes (for tests; default 0).  Takes effect at the
 * next tbsma_build_cells. */
int tbsma_set_tile_box(tbsma_ctx *ctx, int32_t force);

/* Small batches of the shared-memory variant (every tile, or part of a tile, resident on the GPU at once: one wire, a few
 * wires): inside tbsma_md_run's captured step the WHOLE step -- integration, density pass, force pass with the closing
 * kick, per-replica sums, bookkeeping -- is one cooperative kernel with three grid-wide barriers in place of five kernel
 * boundaries (the paper's "+35 % run time due to thread synchronization" between its two stages, is this cost).
 * A step in which a replica needs a new list runs the separate kernels instead (decided on the device).  enable = 0:
 * always the separate kernels.  Default 1.  Changes cost, never results (same operations in the same order), and may be
 * called before or after tbsma_build_cells: how a small batch's tiles are cut into parts (which fixes the grouping of the
 * per-replica sums) does not depend on it. */
int tbsma_set_fused_step(tbsma_ctx *ctx, int32_t enable);
/* 1 if the captured step of tbsma_md_run is that single kernel for the batch as it is now built, else 0. */
int tbsma_get_fused_step(const tbsma_ctx *ctx);

/* Shared-memory variant: how the two gather passes (P:59 stages 1 and 2) are launched.
 *   1 (default) = persistent kernels: two CTAs of 16 warps per SM work through the tiles of the batch, each holding the
 *       image of its NEXT tile while it works on the current one; warps move on to the next tile without a CTA-wide
 *       barrier; the last tiles of a pass are split so that all CTAs finish together;
 *       used for batches of at least four tiles per SM, smaller ones are run as under 0;
 *   2, 3, 4 = persistent kernels whatever the batch size, with that many tile images per CTA (1 uses two);
 *   0 = one CTA per tile (or per 1 / ctas_per_tile of a tile, tbsma_set_tile_split).
 * Changes cost and the grouping of the per-replica fp64 sums, nothing else.  Takes effect at the next tbsma_build_cells. */
int tbsma_set_gather(tbsma_ctx *ctx, int32_t mode);

/* md_run replays one captured step as a CUDA graph when `enable` != 0 (default 2) and the stream is not the legacy
 * default stream.  enable = 2: in the shared-memory variant the kernels that renew cells and candidates (needed in a
 * few steps only, decided on the device) are the body of a conditional IF node of that graph, so that nothing is
 * launched for them otherwise; enable = 1: plain graph, those kernels are launched every step and return at once
 * when there is nothing to do (Nsight Compute cannot profile the kernel nodes of a graph that holds conditional
 * nodes, so profiles are taken with 1); 0: no graph.  Results are identical in all three. */
int tbsma_set_graph(tbsma_ctx *ctx, int32_t enable);

/* Shared-memory variant only.  The list of a replica is renewed in one of two ways: with new cells and candidates
 * (rare, see tbsma_set_outer_skin), ahead of the gather passes of that step; or re-filtered from its candidates.
 * When `enable` (default 1, margin 0.03 A) the second kind is asked for as soon as an atom has moved
 * skin/2 - margin and is written to the second half of the list buffers WHILE the gather passes of the same step
 * still read the previous list (valid until skin/2), on a second stream of the context when
 * tbsma_set_overlap is on; the step's last kernel swaps the halves.  margin must exceed the largest distance an
 * atom moves in one step (0.03 A = 13 sigma_v dt at 298 K, dt = 2 fs); SKIN_VIOLATED is raised if an atom was found
 * beyond skin/2 with its old list still in use.  Off (or margin 0, or a fixed rebuild cadence): every rebuild
 * precedes the gather passes.  Membership of the lists is decided by the predicate of D:A6 either way. */
int tbsma_set_async(tbsma_ctx *ctx, int32_t enable, double margin);

/* Shared-memory variant only: how the asynchronous list renewal above runs beside the gather passes.
 * 2 (default): on `stream` itself, the density pass launched as a PROGRAMMATIC DEPENDENT of the filter kernel (which
 * signals griddepcontrol.launch_dependents at once; the density pass reads the half of the list buffers the filter
 * kernel does not write, and executes griddepcontrol.wait before it exits, so that whatever follows it also follows the
 * filter kernel), so that both run together without a second stream; 1: the filter kernel on a second,
 * high-priority stream of the context, forked and joined inside the step; 0: the same kernels one after the other.
 * The caller sees ordinary stream semantics in all three; results are bitwise identical. */
int tbsma_set_overlap(tbsma_ctx *ctx, int32_t enable);

/* Shared-memory variant: where the records of a tile sit in its shared-memory image.  The gather passes read one
 * 16-byte record per neighbour and lane; eight lanes are served at a time and collide unless their records lie in
 * eight different bank groups (image index mod 8).  The list of every atom is ordered so that they do, as far as the
 * atom's neighbours are spread evenly over the eight groups.  enable = 1 (default): the records get their image index
 * from the COLOUR of the cell of side `cell` (Angstrom; 0 = r0 / sqrt 2, the (100) plane spacing of the fcc crystal the
 * potential describes) their position falls in, (ix + 2 iy + 3 iz) mod 8: on a crystal every neighbourhood then holds
 * nearly equal numbers of each group.  enable = 0: slot order.  Any placement gives the same lists as SETS and the same
 * forces up to the fp32 summation order.  Takes effect when candidates are next rebuilt (tbsma_build_neighbors). */
int tbsma_set_balance(tbsma_ctx *ctx, int32_t enable, double cell);

/* Thermostat of tbsma_md_step / tbsma_md_run.  kind 0 (default): Langevin with the friction passed to those calls
 * (BASELINE.json's substitution).  kind 1: Nose-Hoover, the paper's, which gives neither discretisation nor
 * thermostat mass (D:A17): one variable xi per replica, d xi/dt = (2K - g kB T)/Q, dv/dt = F/m - xi v, Q = g kB T
 * tau_fs^2, g = 3 N_dyn, integrated as B A N A B with N: xi += (dt/2)(2K - g kB T)/Q; v *= exp(-xi dt); K *= s^2;
 * xi += (dt/2)(2K - g kB T)/Q, K the kinetic energy of the dynamic atoms after the opening kick (summed by a kernel of
 * its own at the start of every step, in a fixed order: runs of 256 consecutive atoms by a tree, the runs of a replica in
 * order).  gamma_per_fs and d_seed of the step calls are ignored, d_T is the target.  xi
 * and eta (d eta/dt = xi; E + K + Q xi^2/2 + g kB T eta is conserved) live in the context, start at 0 and are reset by
 * this call and by tbsma_set_system; tbsma_get_thermostat copies them to the host (n_replicas doubles each,
 * synchronises). */
int tbsma_set_thermostat(tbsma_ctx *ctx, int32_t kind, double tau_fs);
int tbsma_get_thermostat(tbsma_ctx *ctx, double *h_xi, double *h_eta);
/* Restores xi and eta (n_replicas doubles each, HOST pointers; synchronises): with pos, vel, force, tag and the step
 * number, which are the caller's, that is the whole state of a Nose-Hoover run.  (The per-replica kinetic energy that drives
 * xi is added in a fixed order, so a run repeats bit for bit; a run resumed in a new context rebuilds its neighbour lists
 * at the restart, i.e. continues with another fp32 summation order: same physics, not the same bits.) */
int tbsma_set_thermostat_state(tbsma_ctx *ctx, const double *h_xi, const double *h_eta);

/* The paper's elongation protocol, beyond the one pulled slab and the constant temperature of tbsma_md_step.
 * All pointers are DEVICE memory owned by the caller and are read at every step until changed; NULL switches a part off.
 *   d_slab1_disp0 / d_slab1_rate (n_replicas doubles each): the OTHER gripping slab (flag 1) moves as well, "the
 *       gripping atoms on the left and right sides of the wire are ... displaced ... in the [-100] and [100] directions"
 *       (P:71): its atoms are PLACED at zref + D1_r, D1_r = disp0_1[r] + rate_1[r] * k, exactly as the flag-2 slab is at
 *       zref + disp0[r] + rate[r] * k (tbsma_md_run; k = steps of the run done, the current one included).  Under
 *       tbsma_md_step k = 1 and rates are NULL, i.e. the caller supplies the total displacements.
 *   stepwise_period P > 0: both slabs move in strokes, "periodically displaced by 0.05 A ... between 20 ps of MD"
 *       (P:71): k is replaced by P * floor(k / P) (paper: P = 10 000 steps of 2 fs, rate * P = +-0.05 A).  0 = every step.
 *   d_T_rate (n_replicas floats, K per step): the target temperature of replica r during step s of a run starting at
 *       step0 is T[r] + T_rate[r] * (s - step0), clamped at 0 ("(2) 400 ps of MD, ramping the temperature from 0.01 K
 *       to the target value"); applies to the Langevin noise and to the Nose-Hoover target alike.
 * NULL protocol = all off (the default). */
typedef struct {
    const double *d_slab1_disp0;
    const double *d_slab1_rate;
    int64_t stepwise_period;
    const float *d_T_rate;
} tbsma_protocol;
int tbsma_set_protocol(tbsma_ctx *ctx, const tbsma_protocol *protocol);

/* Observables of the tensile test as a series recorded ON THE DEVICE inside tbsma_md_run: after
 * every step s with (s + 1) % every == 0 one record of 4 doubles is appended for every replica r at
 * d_series[(r * capacity + d_count[r]) * 4 ...]:
 *     [0] s   [1] strain (Eq.4) = (D2_r - D1_r) / d_L0[r], the displacements of the two slabs at that step
 *     [2] sigma_zz = -(W_zz + K_zz) / d_volume[r] in eV/A^3 (Eq.5 as read in D:A11; z is the wire axis, tension positive;
 *         V is the caller's constant "hard-sphere" volume)
 *     [3] the largest gap (A) between consecutive z coordinates of the replica's atoms (exact when wider than 1/2048 of
 *         the z range the replica's atoms occupy at that step, wherever they are: atoms pulled beyond the box given to
 *         tbsma_set_system count like all others; on a periodic z axis the gap across the boundary is not looked at)
 * and d_count[r] is incremented (the caller zeroes it; recording stops silently at `capacity`).  d_rupture_step[r]
 * (nullable; the caller sets -1) receives the first recorded s whose gap exceeds r_cut: no interaction crosses the gap
 * any more, the wire has parted ("until rupture").  While a series is on, every step evaluates the virial.
 * All pointers are device memory owned by the caller.  NULL series (or every = 0) switches recording off. */
typedef struct {
    int32_t every, capacity;
    double *d_series;
    int32_t *d_count;
    int64_t *d_rupture_step;
    const double *d_volume;
    const double *d_L0;
} tbsma_series;
int tbsma_set_series(tbsma_ctx *ctx, const tbsma_series *series);

/* Stress-strain heat map over all replicas (Fig.4): d_hist[iy * nx + ix] += number of records (k < d_count[r]) of
 * the series whose column col_x (0..3) falls into cell ix of [x_lo, x_hi) cut into nx equal cells and column col_y into
 * cell iy of [y_lo, y_hi) cut into ny; records outside are not counted.  d_hist: nx * ny uint64, accumulated into (the
 * caller zeroes it).  Cell of a value v: floor((v - lo) / (hi - lo) * n) in double. */
int tbsma_series_histogram(tbsma_ctx *ctx, const double *d_series, const int32_t *d_count, int32_t capacity,
                           int32_t col_x, int32_t col_y, double x_lo, double x_hi, int32_t nx, double y_lo, double y_hi,
                           int32_t ny, uint64_t *d_hist, void *stream);

/* Replicas built together (all of them, by tbsma_build_neighbors) that share a temperature would all need their
 * next list at nearly the same step, and again one period later.  When enabled (default 1, more than one replica)
 * replica r rebuilds for the first time as soon as an atom has moved f_r skin/2, f_r = 0.3 + 0.7 frac(0.618 r), and
 * at skin/2 as usual ever after, which spreads the rebuild load evenly over the steps.  Rebuilding early is always
 * valid (D:A14): results change only by the fp32 summation order.  Takes effect at the next tbsma_build_neighbors. */
int tbsma_set_stagger(tbsma_ctx *ctx, int32_t enable);

/* Per-kernel-class timing of tbsma_md_step / tbsma_md_run with CUDA events recorded on the
 * launching stream (graph replay is off while enabled; at most 512 steps are recorded).
 * tbsma_get_timing synchronises on the last event, returns the summed milliseconds of the classes
 * {0 integrate, 1 rebuild chain, 2 density pass, 3 force pass, 4 step bookkeeping} and the number
 * of steps they cover, and resets the record. */
int tbsma_set_timing(tbsma_ctx *ctx, int32_t enable);
int tbsma_get_timing(tbsma_ctx *ctx, double *h_ms_sum5, int64_t *h_steps);

/* Number of this library's kernels launched through ctx since tbsma_set_system (host counter). */
int64_t tbsma_launch_count(const tbsma_ctx *ctx);

const char *tbsma_strerror(int code);
const char *tbsma_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TBSMA_H */
