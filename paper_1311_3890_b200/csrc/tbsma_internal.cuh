// tbsma_internal.cuh -- context layout and launcher declarations shared by the csrc/*.cu files.
// Product code: shares nothing with oracle/.  P:NN = /root/reference/PAPER.md line NN.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "tbsma.h"

#define TBSMA_KB 8.617333262e-5   // eV/K
#define TBSMA_ACC 9.648533212e-3  // 1 eV/(A amu) in A/fs^2

// fp32 constants of the pair functions, folded on the host in double.
// With t = r - r0f (r0f = fl32(r0)):
//   xi^2 exp(-2q x)          = exp2(aq * t + b_rho)
//   (2Ap/r0) exp(-p x)       = exp2(ap * t + b_rep)
//   (q xi^2/r0) exp(-2q x)   = exp2(aq * t + b_band)
struct PairConst {
    float rc2;        // fl32(r_cut)^2 (fp32 product) -- interaction predicate threshold, D:A6
    float rl2;        // fl32(r_cut+skin)^2           -- list predicate threshold
    float ro2;        // fl32(r_cut+skin+outer_skin)^2 -- candidate (outer) list threshold of the tile variant
    float r0f;
    float aq, ap;
    float b_rho, b_rep, b_band;
    float e_rep_scale;  // r0/(2p): sum of (2Ap/r0)e^{-px} -> sum of A e^{-px}
};

// Per-replica geometry (device arrays of R entries).
struct RepGeom {
    float lo[3];
    float len[3];      // fl32(hi - lo): THE box length on periodic axes (D:A6)
    float inv_w[3];    // 1 / cell width
    int nc[3];         // cells per axis
    int cell_base;     // first cell of this replica in the global cell arrays
    int periodic;      // bit a set = axis a periodic
    int atom_begin, atom_end;
};

// One tile of the shared-memory variant: the cells whose atoms one CTA works on ("own") and the cells within one cell of
// them ("halo", own cells included), whose records the CTA stages in shared memory.
//   kind 0: whole z-layers of cells of a thin non-periodic replica (the paper's wires): own layers plus one layer on
//           either side.  Atoms are in cell order (z slowest), so own atoms and halo are CONTIGUOUS slot ranges.
//   kind 1: a box of cells of any replica (thick wires, periodic bulk): the halo is the box grown by one cell per side,
//           wrapped around on periodic axes; every cell is a contiguous run of slots.
// A "run" is a layer (kind 0) or a halo cell (kind 1): the unit inside which atoms are reordered by neighbour count, so
// cell_start stays valid at run boundaries between rebuilds of the cells.
struct TileDesc {
    int rep;          // replica
    int kind;
    int first_of_rep; // the first tile of its replica
    int cell_base;    // first cell of the replica
    int nx, ny, nz;   // cells of the replica per axis
    // kind 0
    int ch0;          // global cell index of the first cell of the first halo layer
    int nlay_h;       // halo layers = own layers + (0..2)
    int own_first;    // index, among the halo layers, of the first own layer (0 or 1)
    int own_n;        // own layers
    int layer_cells;  // nx * ny
    int z_h0;         // z index of the first halo layer
    // kind 1
    short h0[3];      // first halo cell per axis (-1 or nc on a periodic axis: wraps)
    short hn[3];      // halo cells per axis
    short o0[3];      // first own cell per axis, counted from the first halo cell (0 or 1)
    short on[3];      // own cells per axis
    // A tile whose halo wraps around periodic axis a sees a record from across the boundary at a raw coordinate
    // difference beyond half the box: D:A6's `if (d > L/2) d -= L; else if (d < -L/2) d += L` is, for every pair of an own
    // atom and a staged record of THIS tile, `if (|d| > hL[a]) d += Ls[a]` with Ls = -L for a tile at the upper end of the
    // axis, +L at the lower end.  A tile is never at both ends and sees no cell twice because a periodic axis holds at
    // least b + 2 cells for a box of b (tbsma_tile_setup).  With so few cells the two forms can differ in VALUE for pairs
    // more than a cell width w apart (an unwrapped record beyond L/2, which D:A6 would fold back to L - |d| > w), never in
    // the decision: both values exceed w >= r_cut + skin + S.  Every pair that is a member has |d| < w <= L/3 on the near
    // side or L - |d| < w on the far side, where both forms do the same operation.
    float Ls[3], hL[3];   // 0 and +inf on an axis this tile does not wrap
};
// Layout of every neighbour list (int4 rows of the global variant, uint2 rows of the tile variant, candidates too):
// "block-major".  A row is a group of four entries; the rows of the 32 atoms [32 b, 32 b + 32) are contiguous, row g of
// atom i at element tbsma_lrow(i, kg) + 32 g, kg = rows of capacity per atom.  A warp's load of row g is one contiguous
// 256 / 512-byte segment (two if its 32 atoms straddle a block), and ALL rows of a warp's atoms lie within a few KB:
// with the rows of one atom a whole array pitch apart (the first layout) every row of a chunk was in another 2 MB page.
#ifdef __CUDACC__
__host__ __device__ __forceinline__ size_t tbsma_lrow(int i, int kg)
{
    return (size_t)(i >> 5) * ((size_t)kg << 5) + (size_t)(i & 31);
}
#endif
#define TBSMA_LROW 32                // elements between consecutive rows of an atom
#define TBSMA_TILE_MAX_RUNS 128      // halo cells of a box tile
#define TBSMA_TILE_MAX_OWN_RUNS 32
#define TBSMA_TILE_MAX_LAYERS 8      // own layers per tile
#define TBSMA_TILE_MAX_RECORDS 4095  // halo records per tile: (records + sentinel) * 16 B <= 64 KB, u16 byte offsets

// Which replicas a kernel of the rebuild chain works on: replica r takes part iff dirty[r] >= level, and the
// whole launch is a no-op when *any == 0.  dirty[r]: 0 clean, 1 inner list stale, 2 cells + candidate list stale.
struct DirtyView {
    const int *dirty;
    const int *any;
    int level;
};

struct GraphKey {          // arguments a cached one-step CUDA graph was captured with
    const void *p[11];
    double dt, gamma;
    int rebuild_every;
    int epoch;             // tbsma_ctx::epoch when captured: any call that re-sizes, re-allocates or re-tunes bumps it
};

struct tbsma_ctx {
    tbsma_params prm;
    double r_cut, skin;
    PairConst pc;
    int device;
    int n_sm;

    int64_t n;        // atoms
    int n_pad;        // n rounded up to a multiple of 32 (row pitch of the k-major list)
    int R;            // replicas
    int kmax;         // list capacity per atom, multiple of 4
    int64_t n_cells;  // total cells over all replicas
    int any_periodic;
    int variant;        // requested: 0 auto, 1 global gather, 2 shared-memory tiles
    int active_variant; // what the lists are currently built for (1 or 2)
    // tile variant
    int tile_layers;    // own layers per tile requested (<= TBSMA_TILE_MAX_LAYERS)
    int tile_threads;   // CTA size of the tile kernels
    double outer_skin;  // S: the candidate list holds every pair within r_cut + skin + S at its build
    int kmax_o;         // capacity of the candidate list per atom (multiple of 4, <= 248)
    uint2 *d_olist;     // 2 x (kmax_o/4 x n_pad) uint2: candidate list (atom-major rows of kmax_o u16 offsets) + build scratch
    int32_t *d_nn_o;    // n: candidate count | flag << 16
    float4 *d_pos_outer;   // n: positions when the candidate list was built
    int32_t *d_want_outer; // R: the next rebuild of this replica must redo cells + candidate list
    double cell_w;      // cell width the current geometry was computed for
    int tile_cap;       // halo records a tile may hold in shared memory
    int tile_cell_cap;  // halo cells (+1) a tile may hold in shared memory
    int n_tiles;
    TileDesc *d_tiles;
    int32_t *d_tile_first; // R + 1: the tiles of replica r are [first[r], first[r+1])
    int32_t *d_work;       // [0] tiles of replicas with dirty >= 1, [1] with dirty == 2, then the two tile lists
                           // (n_tiles entries each), rebuilt every step by k_tile_worklist
    int own_cap;           // own atoms a tile may hold (sizes the split of the inner build)
    int tile_nsplit;       // CTAs of the gather kernels per tile (> 1 when the tiles are too few to fill the GPU)
    int tile_split_req;    // requested by tbsma_set_tile_split (0 = automatic)
    int tile_force_box;    // tbsma_set_tile_box: box tiles even for replicas whose layers would fit (tests)
    int any_box;           // some replica is cut into box tiles (kind 1)
    int fused_step;        // tbsma_set_fused_step (default 1): small batches run a step as one cooperative kernel
    int fused_max_ctas;    // CTAs of that kernel the GPU holds at once
    int tiles_rejected;    // variant 0: the tiles were tried for this system and the global variant taken instead
    double *d_cta_sums;    // n_tiles x tile_nsplit x 8: E, E_kin, W (xx yy zz xy xz yz) of every CTA of the force pass
    // persistent gather kernels: units = p_plain whole tiles, then the remaining tiles in p_S parts each
    int gather_mode;       // 1 (default): persistent kernels (k_gather_persist); 0: one CTA per tile (or part of a tile)
    int persist_ok;        // two images + sums of a CTA fit half an SM
    int p_S, p_plain, p_units, p_max_chunks;
    int p_tail_split;      // parts the last 2 n_sm tiles of a large batch are cut into (0 = whole)
    int p_nb, p_nb_req;    // tile images per CTA (the next units' images are filled while the current one is worked on)
    size_t have_sums;
    int32_t *d_maxpop;  // 2 R: largest layer population and largest cell population of each replica (measured at build_cells)
    int32_t *d_hbase;   // n: first halo slot of the tile that owns slot i
    int32_t *d_tileof;  // n: the tile that owns slot i
    unsigned short *d_img;  // n_tiles x tile_cap: image index of every halo record of a tile (k_tile_place)
    int32_t *d_inv;         // n_tiles x img_cap: the slot of the record at every image index (inspection calls)
    int img_cap;        // records of a tile image, sentinel and spare room of the colour classes included
    size_t have_tiles, have_first, have_work, have_img, have_inv;   // bytes allocated for the five tile tables
    int balance;        // records placed by colour (default 1) or in slot order
    double class_h;     // side of the colour cells (default r0 / sqrt 2)
    int32_t *d_newslot; // n: cell-order slot -> final slot
    int32_t *d_oldof;   // n: final slot -> cell-order slot
    int32_t *d_nn_tmp;  // n
    float4 *d_tmp_pos;  // n: cell-ordered positions during a rebuild

    // host copies
    int32_t *h_off;
    RepGeom *h_geom;

    // device: topology
    RepGeom *d_geom;        // R
    int32_t *d_atom_rep;    // n: replica of slot i (constant: atoms never change replica)
    // device: cells
    int32_t *d_cell_count;  // n_cells (zero between builds)
    int32_t *d_cell_rep;    // n_cells: replica that owns the cell
    int32_t *d_cell_start;  // n_cells + 1 (global slot of the first atom of each cell)
    int32_t *d_cell_of;     // n
    int32_t *d_slot;        // n
    int32_t *d_order;       // n: new slot -> old slot
    float4 *d_pos_build;    // n: positions at the last build (sorted)
    float4 *d_tmp4;         // n: scratch for the in-place permutation of vel
    int32_t *d_tmp_tag;     // n
    // device: lists
    int32_t *d_nlist;       // n_pad/32 blocks x kmax/4 rows x 32 atoms x int4 (tbsma_lrow): entry k of atom i at
                            // (tbsma_lrow(i, kmax/4) + 32 (k>>2)) * 4 + (k&3)
    int32_t *d_nn;          // n: count | flag<<16
    float4 *d_xs;           // n: (x, y, z, 1/sqrt(rho)) written by the density pass
    // device: control
    int32_t *d_dirty;       // R: replica needs a rebuild
    // Tile variant: list, counts and build positions exist twice (buffer b at offset b * stride of the same
    // allocation).  Replica r reads buffer cur[r]; a rebuild writes the other one and the step's last kernel swaps,
    // so the filter pass of a replica can run beside the gather passes that still use its previous list.
    int list_bufs;          // 1 or 2
    int32_t *d_cur;         // R: buffer in use (all 0 when list_bufs == 1)
    int async_inner;        // enabled (default 1): see tbsma_set_async
    double async_margin;    // A: the list is renewed once an atom has moved skin/2 - margin
    float *d_stagger;       // R: factor on (skin/2)^2 until the replica's first rebuild (spreads the rebuilds of
                            // replicas that start together over the steps); 1 afterwards
    int stagger;            // enabled (default 1)
    int32_t *d_ctrl;        // [0] any replica dirty, [1] status flags, [2] max neighbours seen, [3] any dirty == 2,
                            // [4] / [5] next unit of the persistent density / force pass (k_gather_persist; zeroed ahead of
                            // every density pass by k_tile_worklist or a memset, and by the opposite pass), [6..7] unused
    unsigned long long *d_counters; // [0] step offset inside md_run, [1] replica builds, [2] build passes, [3] steps,
                                    // [4..5] count_pairs scratch, [6] replica builds that redid cells + candidates,
                                    // [7] step number of the first step of the md_run in flight (captured steps read it)
    // host staging for *_host entry point
    float4 *s_pos, *s_vel, *s_force;
    int32_t *s_tag;
    float *s_T;
    unsigned long long *s_seed;
    double *s_disp0, *s_rate, *s_e, *s_w, *s_k;
    int64_t s_n;
    int s_R;

    // Nose-Hoover thermostat (the paper's; tbsma_set_thermostat): one variable per replica
    int thermostat_kind;       // 0 Langevin (gamma of tbsma_md_step), 1 Nose-Hoover
    double nh_tau;             // fs: Q = g kB T tau^2
    double *d_nh;              // 2 R: xi, eta
    double *d_kmid;            // 2 n_blk: kinetic energy after the opening kick and number of dynamic atoms of every run
                               // of 256 consecutive atoms of a replica
    int32_t *d_blk_rep;        // n_blk: replica of the run
    int32_t *d_blk_first;      // R + 1: first run of every replica
    int n_blk;
    float *d_nh_scale;         // R
    // the paper's elongation protocol (tbsma_set_protocol) and its observables as a device-side series
    // (tbsma_set_series)
    tbsma_protocol proto;
    tbsma_series series;       // every == 0: off
    double *d_series_w;        // R x 6: virial of the step when the caller of tbsma_md_run passes none
    int cells_built, list_built;
    int epoch;                 // bumped by every call after which a captured step would hold stale arguments
    int64_t launches;
    // md_run: one step captured as a CUDA graph and replayed
    int use_graph;
    cudaGraphExec_t graph_exec;
    cudaGraphExec_t graph_exec_multi;   // graph_multi_steps steps in one graph (small batches)
    int graph_multi_steps;
    GraphKey graph_key;
    int64_t graph_launches_per_step;
    cudaStream_t own_stream;   // used by the *_host entry point
    // md step of the tile variant: rebuild chain + rebuilt replicas on a second (high-priority) stream
    int overlap;               // enabled (default 1)
    cudaStream_t aux_stream;
    cudaStream_t body_stream;  // captures the body of the conditional node of a captured step
    int use_cond;              // captured steps wrap the cells + candidates chain in an IF node (default 1)
    cudaEvent_t ev_fork, ev_join;
    // optional per-kernel-class timing with CUDA events on the launching stream
    int timing;
    cudaEvent_t *tev;          // 6 events per timed step (class boundaries)
    int tev_steps;             // steps recorded so far
};
#define TBSMA_TIMING_MAX_STEPS 512

// ---- launchers (each returns cudaError_t of the launch) -------------------------------------
// cells / lists (tbsma_cells.cu)
cudaError_t tbsma_launch_rebuild(tbsma_ctx *c, float4 *pos, float4 *vel, int32_t *tag, bool do_cells,
                                 bool do_list, cudaStream_t st);
cudaError_t tbsma_launch_mark_all_dirty(tbsma_ctx *c, cudaStream_t st);
inline DirtyView tbsma_dirty_view(const tbsma_ctx *c)
{
    DirtyView v;
    v.dirty = c->d_dirty;
    v.level = c->active_variant == 2 ? 2 : 1;
    v.any = c->d_ctrl + (v.level == 2 ? 3 : 0);
    return v;
}
cudaError_t tbsma_launch_get_neighbors(tbsma_ctx *c, const int32_t *tag, int32_t *counts, int32_t *list,
                                       cudaStream_t st);
// a6 in the tile variant: per-replica sums from the sums the CTAs of the force pass left, in tile order
struct TileSums {
    const double *cta_sums;   // nullptr: nothing to do
    const int *tile_first;    // R + 1
    int nsplit;
    double *e_rep, *ekin, *w_rep;   // each nullable
};
#ifdef __CUDACC__
// Called by all threads of every CTA of a grid of tbsma_reduce_grid(R) CTAs of 256 threads.  Many replicas: a warp per
// replica, lane l adds the replica's CTAs l, l + 32, ... in order and a shuffle tree adds the lanes.  Few replicas (one
// long wire has thousands of tiles): CTA 0 takes one replica at a time, thread t adds CTAs t, t + 256, ... and a fixed
// tree adds the threads.  Either way the order is fixed: bitwise repeatable.
inline int tbsma_reduce_grid(int R) { return R >= 64 ? (R + 7) / 8 : 1; }
__device__ inline void tbsma_reduce_replicas(const TileSums &ts, int R)
{
    if (!ts.cta_sums) return;
    const int nq = ts.w_rep ? 8 : 2;
    if (R >= 64) {
        const int r = (int)blockIdx.x * 8 + (int)(threadIdx.x >> 5), lane = threadIdx.x & 31;
        if (r >= R) return;
        double acc[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        const int j0 = ts.tile_first[r] * ts.nsplit, j1 = ts.tile_first[r + 1] * ts.nsplit;
        for (int j = j0 + lane; j < j1; j += 32) {
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (q < nq) acc[q] += ts.cta_sums[8 * (size_t)j + q];
        }
#pragma unroll
        for (int q = 0; q < 8; ++q)
            for (int o = 16; o > 0; o >>= 1) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
        if (lane == 0) {
            if (ts.e_rep) ts.e_rep[r] = acc[0];
            if (ts.ekin) ts.ekin[r] = acc[1];
            if (ts.w_rep)
                for (int q = 0; q < 6; ++q) ts.w_rep[6 * (size_t)r + q] = acc[2 + q];
        }
        return;
    }
    if (blockIdx.x != 0) return;
    __shared__ double red[8][256];
    for (int r = 0; r < R; ++r) {
        double acc[8] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        const int j0 = ts.tile_first[r] * ts.nsplit, j1 = ts.tile_first[r + 1] * ts.nsplit;
        // (unrolled over the eight quantities with a guard: a run-time index would put acc[] into local memory)
        for (int j = j0 + (int)threadIdx.x; j < j1; j += 256) {
#pragma unroll
            for (int q = 0; q < 8; ++q)
                if (q < nq) acc[q] += ts.cta_sums[8 * (size_t)j + q];
        }
        __syncthreads();
#pragma unroll
        for (int q = 0; q < 8; ++q) red[q][threadIdx.x] = acc[q];
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if ((int)threadIdx.x < o) {
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    if (q < nq) red[q][threadIdx.x] += red[q][threadIdx.x + o];
            }
            __syncthreads();
        }
        if (threadIdx.x == 0) {
            if (ts.e_rep) ts.e_rep[r] = red[0][0];
            if (ts.ekin) ts.ekin[r] = red[1][0];
            if (ts.w_rep)
                for (int q = 0; q < 6; ++q) ts.w_rep[6 * (size_t)r + q] = red[2 + q][0];
        }
    }
}
#endif

#ifdef __CUDACC__
// end of a step, by all threads of ONE CTA: statistics, clear the dirty flags, swap the list halves of the replicas that
// were rebuilt, advance the in-run step offset (k_finish_step; the fused step kernel of small batches)
__device__ inline void tbsma_finish_bookkeeping(int *__restrict__ dirty, int *__restrict__ ctrl, float *__restrict__ stagger,
                                                int *__restrict__ cur, int swap, unsigned long long *__restrict__ counters,
                                                int R, int advance, int count_step)
{
    __shared__ int s_cnt, s_cnt2;
    if (threadIdx.x == 0) { s_cnt = 0; s_cnt2 = 0; }
    __syncthreads();
    if (ctrl[0]) {
        int mine = 0, mine2 = 0;
        for (int r = threadIdx.x; r < R; r += blockDim.x) {
            const int d = dirty[r];
            if (d) { ++mine; dirty[r] = 0; stagger[r] = 1.0f; if (swap) cur[r] ^= 1; }
            if (d == 2) ++mine2;
        }
        if (mine) atomicAdd(&s_cnt, mine);
        if (mine2) atomicAdd(&s_cnt2, mine2);
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (ctrl[0]) {
            counters[1] += (unsigned long long)s_cnt; counters[2] += 1ull; counters[6] += (unsigned long long)s_cnt2;
            ctrl[0] = 0; ctrl[3] = 0;
        }
        if (count_step) counters[3] += 1ull;
        if (advance) counters[0] += 1ull;
    }
}
#endif

// forces (tbsma_force.cu)
struct KickArgs {
    float4 *vel;          // nullptr = no fused half kick
    float kick;           // (dt/2) c/m
    float ke_scale;       // m/(2c)
    double *ekin;         // per replica, nullable
};
cudaError_t tbsma_launch_density(tbsma_ctx *c, const float4 *pos, cudaStream_t st);
cudaError_t tbsma_launch_force(tbsma_ctx *c, float4 *force, double *e_rep, double *w_rep, KickArgs kick,
                               cudaStream_t st);
cudaError_t tbsma_launch_count_pairs(tbsma_ctx *c, const float4 *pos, unsigned long long *d_out2,
                                     cudaStream_t st);
// shared-memory tile variant (tbsma_tile.cu)
int tbsma_tile_setup(tbsma_ctx *c, cudaStream_t st);   // host: sizes the tiles from the binned cells (synchronises)
cudaError_t tbsma_launch_tile_lists(tbsma_ctx *c, float4 *pos, float4 *vel, int32_t *tag, cudaStream_t st);
// tiles of the dirty replicas, from the flags; use_cond: also sets the graph conditional `cond` (any replica with dirty == 2)
cudaError_t tbsma_launch_tile_worklist(tbsma_ctx *c, cudaStream_t st, unsigned long long cond = 0ull, int use_cond = 0);
// inner lists of the replicas on work list `which` (0: dirty == 1, 1: dirty == 2), written to the buffer not in use
cudaError_t tbsma_launch_tile_inner(tbsma_ctx *c, const float4 *pos, int which, cudaStream_t st, bool beside = false);
cudaError_t tbsma_launch_stage_copy(tbsma_ctx *c, const float4 *pos, const float4 *vel, const int32_t *tag,
                                    cudaStream_t st);
// sync_level: the gather passes read the freshly written half of the list buffers for replicas with
// dirty >= sync_level (their rebuild ran ahead of the launch), the half in use for all others.
cudaError_t tbsma_launch_density_tile(tbsma_ctx *c, const float4 *pos, int sync_level, cudaStream_t st,
                                      bool early = false);
// leaves the sums of every CTA in d_cta_sums (virial: with W); per-replica sums by tbsma_launch_reduce_replicas or,
// inside an MD step, by k_finish_step
cudaError_t tbsma_launch_force_tile(tbsma_ctx *c, float4 *force, bool virial, KickArgs kick, int sync_level,
                                    cudaStream_t st);
TileSums tbsma_tile_sums(const tbsma_ctx *c, double *e_rep, double *ekin, double *w_rep);
struct StepArgs;
bool tbsma_step_small_ok(const tbsma_ctx *c);
cudaError_t tbsma_launch_step_small(tbsma_ctx *c, float4 *pos, float4 *vel, float4 *force, const int32_t *tag,
                                    const StepArgs &a, KickArgs kick, bool virial, int advance_offset, TileSums ts,
                                    unsigned long long cond, cudaStream_t st);
cudaError_t tbsma_launch_reduce_replicas(tbsma_ctx *c, double *e_rep, double *ekin, double *w_rep, cudaStream_t st);
cudaError_t tbsma_launch_get_neighbors_tile(tbsma_ctx *c, const int32_t *tag, int32_t *counts, int32_t *list,
                                            cudaStream_t st);
cudaError_t tbsma_launch_count_pairs_tile(tbsma_ctx *c, const float4 *pos, unsigned long long *d_out2,
                                          cudaStream_t st);
// integrator (tbsma_integrate.cu)
struct StepArgs {
    float half_dt, kick, c1, c2, sigma_scale;  // sigma_v = sigma_scale * sqrt(T)
    float skin_half2;        // (skin/2)^2: beyond it the list in use is no longer guaranteed
    float trigger2;          // displacement^2 that asks for a new list (= skin_half2 unless lists are renewed one step late)
    const int *cur;          // per replica: which half of pos_build belongs to the list in use
    int pb_stride;           // float4 elements between the two halves of pos_build
    int thermostat;          // gamma > 0
    int rebuild_every;
    unsigned long long step_base;
    int step_on_device;      // the step number of the run's first step is d_counters[7], not step_base (captured steps)
    const float *T;
    const unsigned long long *seed;
    const double *disp0;     // nullable
    const double *rate;      // nullable
    const int *want_outer;   // nullable (tile variant): replicas whose next rebuild redoes cells + candidates
    const float *stagger;    // per replica factor on skin_half2
    const float *nh_scale;   // nullable: Nose-Hoover velocity scale of this step per replica (replaces the O part)
    const double *disp0_1;   // nullable: the flag-1 slab (both ends are displaced), as disp0 / rate for the flag-2 slab
    const double *rate_1;    // nullable
    long long period;        // > 0: the slabs advance every `period` steps by period x rate ("periodically displaced")
    const float *T_rate;     // nullable: target temperature of replica r during step s is T[r] + T_rate[r] (s - step0)
    double *e_rep, *w_rep, *ekin;  // zeroed here for the force pass; nullable
};
cudaError_t tbsma_launch_integrate_pre(tbsma_ctx *c, float4 *pos, float4 *vel, const float4 *force,
                                       const int32_t *tag, const StepArgs &a, cudaStream_t st);
cudaError_t tbsma_launch_finish_step(tbsma_ctx *c, int advance_offset, cudaStream_t st, TileSums ts = TileSums());
cudaError_t tbsma_launch_set_stagger(tbsma_ctx *c, cudaStream_t st);
cudaError_t tbsma_launch_set_step_base(tbsma_ctx *c, unsigned long long step0, cudaStream_t st);
cudaError_t tbsma_launch_nose_hoover(tbsma_ctx *c, const float4 *pos, const float4 *vel, const float4 *force,
                                     const StepArgs &a, double dt, cudaStream_t st);
// after the last kernel of a step of tbsma_md_run: appends a record to the series of every replica when one is due
cudaError_t tbsma_launch_series_record(tbsma_ctx *c, const float4 *pos, const float4 *vel, const double *w_rep,
                                       const StepArgs &a, cudaStream_t st);
cudaError_t tbsma_launch_series_histogram(tbsma_ctx *c, const double *series, const int32_t *count, int capacity, int col_x,
                                          int col_y, double x_lo, double x_hi, int nx, double y_lo, double y_hi, int ny,
                                          unsigned long long *hist, cudaStream_t st);
cudaError_t tbsma_launch_kinetic_tensor(tbsma_ctx *c, const float4 *pos, const float4 *vel, double *k_rep, cudaStream_t st);
cudaError_t tbsma_launch_stress(tbsma_ctx *c, const double *w_rep, const double *k_rep, const double *volume,
                                double *sigma, cudaStream_t st);
