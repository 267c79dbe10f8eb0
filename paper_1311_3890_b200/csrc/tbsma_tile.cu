// tbsma_tile.cu -- the shared-memory variant of the neighbour machinery and of the two neighbour-gather passes (SURVEY
// rows a2, a3, a4, a6): layer tiles for thin wires (below), box tiles for thick wires and periodic replicas (TileDesc,
// TileMap), persistent gather kernels for large batches (k_gather_persist), the whole step as one cooperative kernel
// for small ones (k_step_small).
//
// The paper's systems are thin [100] wires and its best performance came with the
// atoms ordered along the wire axis.  With cells numbered z-slowest, a run of z-layers of
// cells ("tile") and its one-layer halo are CONTIGUOUS index ranges, so one CTA can stage every
// position its atoms will ever gather (a few thousand records) in shared memory with one coalesced
// read of the range and serve all neighbour gathers from there.  That allows
//   * 16-bit neighbour entries (byte offsets into the tile's shared-memory image): half the list
//     bytes of the int32 list, which is the dominant HBM stream of both passes;
//   * atoms ordered inside each layer by neighbour count (longest lists first), so the 32 lanes of
//     a warp run the same number of iterations (surface atoms of a 3 nm wire have 42 partners,
//     core atoms 86);
//   * each atom's list ordered so that at step p lane l reads a record of bank group (l + p) mod 8:
//     the eight lanes served by one shared-memory wavefront of a 128-bit load then hit eight
//     different 16-byte bank groups (summation order is free, A15);
//   * the records placed in the image by the colour of a spatial hash (k_tile_place), so that every
//     atom's neighbours are spread evenly over the eight bank groups and that order has few holes.
// Membership is the fp32 predicate of D:A6, operation for operation, as in tbsma_cells.cu.
//
// Two-level lists.  Scanning 27 cells costs about five force passes per atom, and at 298 K a replica
// needs a fresh list every ~12 steps (fewer rebuilds are why 10 K runs faster).  So the cell
// scan builds a CANDIDATE list with the larger radius r_cut + skin + S (S = outer_skin, 2.5 A by default):
// K1 (scan), K1b (place), K2 (finish), K3 (permute) below, rarely.  The list the gather passes read
// (radius r_cut + skin, the paper's r_buff list) is filtered from the candidates by the tile that
// owns the atom (k_tile_inner) when the replica's atoms have moved skin/2 (less a margin when the filter
// pass runs beside the gather passes, tbsma_set_async): ~2.7 candidates per kept entry instead of ~9.
// A candidate list stays valid while no atom moved more than S/2 since it was built; the inner build
// checks that (status flag) and asks for new candidates one rebuild earlier (want_outer).  Slots (and
// so the u16 offsets) only change when candidates are rebuilt.  The list, its counts and its build
// positions exist twice (ListSel): a renewal writes the half not in use, the step's last kernel swaps.
#include <cooperative_groups.h>

#include "tbsma_integrate.cuh"

namespace {

constexpr int kScanThreads = 1024;  // k_tile_scan: one round for tiles of <= 1024 own atoms (the rebuild chain is
                                    // latency bound: only the dirty replicas' tiles do any work)
constexpr int kFinishMaxThreads = 1024;

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// index ranges of a tile, from the cell starts at its layer boundaries
struct TileRange { int halo_lo, nh, lo, hi; };
__device__ __forceinline__ TileRange tile_range(const TileDesc &t, const int *__restrict__ cell_start)
{
    TileRange r;
    r.halo_lo = cell_start[t.ch0];
    r.nh = cell_start[t.ch0 + t.nlay_h * t.layer_cells] - r.halo_lo;
    r.lo = cell_start[t.ch0 + t.own_first * t.layer_cells];
    r.hi = cell_start[t.ch0 + (t.own_first + t.own_n) * t.layer_cells];
    return r;
}

// Runs of a tile (layers or halo cells, see TileDesc) in shared memory: where every halo record and every own atom lives.
// Halo-local index k = position among the tile's staged records, runs concatenated in order; own-local index o = position
// among the tile's own atoms, own runs concatenated in order.  Lane o & 31 handles atom o in the list builds and in the
// gather passes alike (the bank schedule of the lists depends on it).
struct TileMap {
    int n_runs, nh, n_own_runs, n_own;
    int contig;                            // layer tiles: halo and own atoms are contiguous slot ranges (no search)
    int own_slot0;                         // slot of own-local index 0
    int lstart[TBSMA_TILE_MAX_RUNS + 1];   // halo-local index of the first record of run r; lstart[n_runs] = nh
    int gslot[TBSMA_TILE_MAX_RUNS];        // slot of that record
    int ostart[TBSMA_TILE_MAX_OWN_RUNS + 1];   // own-local index of the first atom of own run q
    short orun[TBSMA_TILE_MAX_OWN_RUNS];       // which run it is
};
__device__ __forceinline__ int wrap_cell(int c, int nc) { return c < 0 ? c + nc : (c >= nc ? c - nc : c); }

// called by every thread of the CTA; ends with a barrier
__device__ __forceinline__ void tile_map_build(const TileDesc &t, const int *__restrict__ cell_start, TileMap &M)
{
    if (t.kind == 0) {       // a handful of layers: one thread, one barrier
        if (threadIdx.x == 0) {
            const int base = cell_start[t.ch0];
            M.lstart[0] = 0;
            for (int r = 0; r < t.nlay_h; ++r) {
                const int s = r == 0 ? base : M.gslot[r - 1] + (M.lstart[r] - M.lstart[r - 1]);
                const int e = cell_start[t.ch0 + (r + 1) * t.layer_cells];
                M.gslot[r] = s;
                M.lstart[r + 1] = e - base;
            }
            M.n_runs = t.nlay_h;
            M.nh = M.lstart[t.nlay_h];
            int o = 0;
            for (int l = 0; l < t.own_n; ++l) {
                const int r = t.own_first + l;
                M.orun[l] = (short)r; M.ostart[l] = o; o += M.lstart[r + 1] - M.lstart[r];
            }
            M.ostart[t.own_n] = o;
            M.n_own_runs = t.own_n;
            M.n_own = o;
            M.contig = 1;
            M.own_slot0 = M.gslot[t.own_first];
        }
        __syncthreads();
        return;
    }
    const int n_runs = t.kind == 0 ? t.nlay_h : (int)t.hn[0] * t.hn[1] * t.hn[2];
    for (int r = threadIdx.x; r < n_runs; r += blockDim.x) {
        int c0, nc;
        if (t.kind == 0) {
            c0 = t.ch0 + r * t.layer_cells;
            nc = t.layer_cells;
        } else {
            const int hx = r % t.hn[0], hy = (r / t.hn[0]) % t.hn[1], hz = r / (t.hn[0] * t.hn[1]);
            const int cx = wrap_cell(t.h0[0] + hx, t.nx), cy = wrap_cell(t.h0[1] + hy, t.ny), cz = wrap_cell(t.h0[2] + hz, t.nz);
            c0 = t.cell_base + (cz * t.ny + cy) * t.nx + cx;
            nc = 1;
        }
        const int s = cell_start[c0];
        M.gslot[r] = s;
        M.lstart[r + 1] = cell_start[c0 + nc] - s;       // population, made a prefix sum below
    }
    __syncthreads();
    if (threadIdx.x < 32) {          // inclusive scan of the populations by one warp, 32 runs per round
        const int lane = threadIdx.x;
        int carry = 0;
        for (int r0 = 0; r0 < n_runs; r0 += 32) {
            int v = r0 + lane < n_runs ? M.lstart[r0 + lane + 1] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, v, o);
                if (lane >= o) v += y;
            }
            if (r0 + lane < n_runs) M.lstart[r0 + lane + 1] = carry + v;
            carry += __shfl_sync(0xffffffffu, v, 31);
        }
        if (lane == 0) { M.lstart[0] = 0; M.n_runs = n_runs; M.nh = carry; }
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        int q = 0, o = 0;
        if (t.kind == 0) {
            for (int l = 0; l < t.own_n; ++l) {
                const int r = t.own_first + l;
                M.orun[q] = (short)r; M.ostart[q] = o; o += M.lstart[r + 1] - M.lstart[r]; ++q;
            }
        } else {
            for (int z = 0; z < t.on[2]; ++z)
                for (int y = 0; y < t.on[1]; ++y)
                    for (int x = 0; x < t.on[0]; ++x) {
                        const int r = ((t.o0[2] + z) * t.hn[1] + t.o0[1] + y) * t.hn[0] + t.o0[0] + x;
                        M.orun[q] = (short)r; M.ostart[q] = o; o += M.lstart[r + 1] - M.lstart[r]; ++q;
                    }
        }
        M.ostart[q] = o;
        M.n_own_runs = q;
        M.n_own = o;
        M.contig = 0;
        M.own_slot0 = 0;
    }
    __syncthreads();
}
// run that holds halo-local index k (< nh)
__device__ __forceinline__ int map_run_of(const TileMap &M, int k)
{
    int lo = 0, hi = M.n_runs - 1;
    while (lo < hi) {
        const int mid = (lo + hi + 1) >> 1;
        if (M.lstart[mid] <= k) lo = mid; else hi = mid - 1;
    }
    return lo;
}
__device__ __forceinline__ int map_slot(const TileMap &M, int k)
{
    if (M.contig) return M.gslot[0] + k;
    const int r = map_run_of(M, k);
    return M.gslot[r] + k - M.lstart[r];
}
// own-local index o (< n_own) -> slot; also its own run q and its halo-local index
__device__ __forceinline__ int map_own(const TileMap &M, int o, int &q, int &k)
{
    q = 0;
    while (q + 1 < M.n_own_runs && M.ostart[q + 1] <= o) ++q;
    const int r = M.orun[q], off = o - M.ostart[q];
    k = M.lstart[r] + off;
    return M.gslot[r] + off;
}
__device__ __forceinline__ int map_own(const TileMap &M, int o)
{
    if (M.contig) return M.own_slot0 + o;
    int q, k;
    return map_own(M, o, q, k);
}
// D:A6 for a pair of an own atom and a staged record of a tile that wraps around periodic axes (see TileDesc)
__device__ __forceinline__ float wrap_d(float d, float hL, float Ls) { return fabsf(d) > hL ? d + Ls : d; }

// largest layer population of every replica (sizes the tiles; host reads it back at build_cells)
__global__ void k_layer_maxpop(const RepGeom *__restrict__ geom, const int *__restrict__ cell_start,
                               int *__restrict__ maxpop, int R)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    const RepGeom *g = geom + r;
    const int lc = g->nc[0] * g->nc[1];
    int m = 0;
    for (int z = 0; z < g->nc[2]; ++z)
        m = max(m, cell_start[g->cell_base + (z + 1) * lc] - cell_start[g->cell_base + z * lc]);
    maxpop[r] = m;
    int mc = 0;        // and the largest cell population (sizes box tiles)
    const int ncell = lc * g->nc[2];
    for (int c = 0; c < ncell; ++c) mc = max(mc, cell_start[g->cell_base + c + 1] - cell_start[g->cell_base + c]);
    maxpop[R + r] = mc;
}

// ---- worklists.  Only a few per cent of the replicas rebuild in a given step, so the kernels that
// work on them loop over a list of their tiles instead of launching one (mostly idle) CTA per tile.
// work[0] = tiles of replicas with dirty == 1 (new list from the old candidates), work[1] = with dirty == 2
// (new cells and candidates first), then the two tile lists.
__global__ void __launch_bounds__(256)
k_tile_worklist(const int *__restrict__ dirty, const int *__restrict__ tile_first, int *__restrict__ work, int R,
                int n_tiles, cudaGraphConditionalHandle cond, int use_cond, int *__restrict__ claims)
{
    __shared__ int s_base[2], s_warp[2][8];
    // unit counters of the persistent gather passes of this step (ctrl[4..5]): they start every step at zero whatever the
    // step before left behind (a pass that was launched without its partner, a launch that failed)
    if (threadIdx.x < 2) { s_base[threadIdx.x] = 0; claims[threadIdx.x] = 0; }
    __syncthreads();
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    for (int r0 = 0; r0 < R; r0 += 256) {
        const int r = r0 + threadIdx.x;
        const int d = r < R ? dirty[r] : 0;
        const int f = r < R ? tile_first[r] : 0, nt = r < R ? tile_first[r + 1] - f : 0;
        int v[2] = {d == 1 ? nt : 0, d == 2 ? nt : 0}, incl[2];
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            int x = v[k];
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int y = __shfl_up_sync(0xffffffffu, x, o);
                if (lane >= o) x += y;
            }
            incl[k] = x;
            if (lane == 31) s_warp[k][wid] = x;
        }
        __syncthreads();
#pragma unroll
        for (int k = 0; k < 2; ++k) {
            int off = s_base[k];
            for (int w = 0; w < wid; ++w) off += s_warp[k][w];
            int *dst = work + 2 + k * n_tiles + off + incl[k] - v[k];
            for (int q = 0; q < v[k]; ++q) dst[q] = f + q;
        }
        __syncthreads();
        if (threadIdx.x < 2) {
            int tot = 0;
            for (int w = 0; w < 8; ++w) tot += s_warp[threadIdx.x][w];
            s_base[threadIdx.x] += tot;
        }
        __syncthreads();
    }
    if (threadIdx.x < 2) work[threadIdx.x] = s_base[threadIdx.x];
    // inside a captured step the cells + candidates chain is the body of an IF node: skipped unless a replica needs it
    if (use_cond && threadIdx.x == 0) cudaGraphSetConditional(cond, s_base[1] > 0 ? 1u : 0u);
}

// ---- K1: scan.  Cell-ordered positions of the tile + halo in shared memory; every own atom scans
// its 3 x 3 runs of x-adjacent cells, writes its partners (halo-local cell-order indices, u16) to
// the temporary list, and is ranked inside its layer by (count descending, slot ascending).
struct ScanArgs {
    const int *cell_start, *cell_sorted;
    int *ctrl;
    const float4 *pos_sorted;
    uint2 *nl_tmp;
    int *nn_tmp, *newslot, *oldof, *want_outer;
    int n_pad, kmax;
    float ro2, rl2;
    int s_cap, cell_cap;
};

__device__ __forceinline__ void scan_tile(const TileDesc &t, const ScanArgs &A)
{
    const int *__restrict__ cell_start = A.cell_start;
    const int *__restrict__ cell_sorted = A.cell_sorted;
    int *__restrict__ ctrl = A.ctrl;
    const float4 *__restrict__ pos_sorted = A.pos_sorted;
    uint2 *__restrict__ nl_tmp = A.nl_tmp;
    int *__restrict__ nn_tmp = A.nn_tmp, *__restrict__ newslot = A.newslot, *__restrict__ oldof = A.oldof;
    int *__restrict__ want_outer = A.want_outer;
    const int n_pad = A.n_pad, kmax = A.kmax, s_cap = A.s_cap, cell_cap = A.cell_cap;
    const float ro2 = A.ro2, rl2 = A.rl2;
    if (threadIdx.x == 0 && t.first_of_rep) want_outer[t.rep] = 0;   // new candidates: request served
    extern __shared__ float4 smem_f4[];
    float4 *sm = smem_f4;
    int *cs = reinterpret_cast<int *>(sm + s_cap);
    unsigned short *cnts = reinterpret_cast<unsigned short *>(cs + cell_cap);
    __shared__ int lb[TBSMA_TILE_MAX_LAYERS + 4];
    const int tid = threadIdx.x;
    if (tid <= t.nlay_h) lb[tid] = cell_start[t.ch0 + tid * t.layer_cells];
    __syncthreads();
    const int halo_lo = lb[0], nh = lb[t.nlay_h] - halo_lo;
    const int lo = lb[t.own_first], hi = lb[t.own_first + t.own_n];
    if (hi <= lo) return;
    if (nh > s_cap) {
        if (tid == 0) atomicOr(ctrl + 1, (int)TBSMA_FLAG_TILE_OVERFLOW);
        return;
    }
    const int ncell_h = t.nlay_h * t.layer_cells;
    for (int k = tid; k <= ncell_h; k += blockDim.x) cs[k] = cell_start[t.ch0 + k] - halo_lo;
    for (int k = tid; k < nh; k += blockDim.x) sm[k] = pos_sorted[halo_lo + k];
    __syncthreads();
    const int nx = t.nx, ny = t.ny, nz = t.nz;
    for (int a = lo + tid; a < hi; a += blockDim.x) {
        const int al = a - halo_lo;
        const float4 pi = sm[al];
        const int lc = cell_sorted[a] - t.cell_base;
        const int cx = lc % nx, cy = (lc / nx) % ny, cz = lc / t.layer_cells;
        const int x0 = max(cx - 1, 0), x1 = min(cx + 1, nx - 1);
        uint2 *row = nl_tmp + tbsma_lrow(a, kmax >> 2);
        unsigned w0 = 0u, w1 = 0u;
        int cnt = 0, cnt_in = 0;     // candidates (d2 < ro2) and list members (d2 < rl2, orders the layer)
        for (int zz = max(cz - 1, 0); zz <= min(cz + 1, nz - 1); ++zz)
            for (int yy = max(cy - 1, 0); yy <= min(cy + 1, ny - 1); ++yy) {
                const int cb = ((zz - t.z_h0) * ny + yy) * nx;
                const int s = cs[cb + x0], e = cs[cb + x1 + 1];
                for (int j = s; j < e; ++j) {
                    const float4 pj = sm[j];
                    const float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
                    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));   // D:A6
                    if (d2 < ro2 && j != al) {
                        if (cnt < kmax) {
                            const unsigned v = (unsigned)j << ((cnt & 1) << 4);
                            if (cnt & 2) w1 |= v; else w0 |= v;
                            if ((cnt & 3) == 3) {
                                row[(size_t)(cnt >> 2) * TBSMA_LROW] = make_uint2(w0, w1);
                                w0 = w1 = 0u;
                            }
                        }
                        ++cnt;
                        cnt_in += d2 < rl2;
                    }
                }
            }
        if (cnt > kmax) atomicOr(ctrl + 1, (int)TBSMA_FLAG_NLIST_OVERFLOW);
        cnt = min(cnt, kmax);
        if (cnt & 3) row[(size_t)(cnt >> 2) * TBSMA_LROW] = make_uint2(w0, w1);
        cnts[a - lo] = (unsigned short)cnt_in;
        nn_tmp[a] = cnt | ((__float_as_int(pi.w) & 3) << 16);
    }
    __syncthreads();
    for (int a = lo + tid; a < hi; a += blockDim.x) {
        int m = t.own_first;
        while (a >= lb[m + 1]) ++m;
        const int l0 = lb[m] - lo, l1 = lb[m + 1] - lo, me = a - lo;
        const int my = cnts[me];
        int rank = 0;
        for (int b = l0; b < l1; ++b) {
            const int cb = cnts[b];
            rank += (cb > my) || (cb == my && b < me);
        }
        const int ns = lb[m] + rank;
        newslot[a] = ns;
        oldof[ns] = a;
    }
}

// K1 for a box tile (kind 1): the same scan over the 3 x 3 runs of x-adjacent halo cells, pair differences wrapped as
// D:A6 prescribes where the tile's halo wraps around a periodic axis; ranks inside the own CELL.
__device__ __forceinline__ void scan_box(const TileDesc &t, const ScanArgs &A)
{
    extern __shared__ float4 smem_f4[];
    float4 *sm = smem_f4;
    unsigned short *cnts = reinterpret_cast<unsigned short *>(sm + A.s_cap);
    __shared__ TileMap M;
    const int tid = threadIdx.x;
    if (tid == 0 && t.first_of_rep) A.want_outer[t.rep] = 0;   // new candidates: request served
    tile_map_build(t, A.cell_start, M);
    if (M.n_own <= 0) return;
    if (M.nh > A.s_cap) {
        if (tid == 0) atomicOr(A.ctrl + 1, (int)TBSMA_FLAG_TILE_OVERFLOW);
        return;
    }
    for (int k = tid; k < M.nh; k += blockDim.x) sm[k] = A.pos_sorted[map_slot(M, k)];
    __syncthreads();
    const int hn0 = t.hn[0], hn1 = t.hn[1], hn2 = t.hn[2];
    const float hLx = t.hL[0], hLy = t.hL[1], hLz = t.hL[2], Lsx = t.Ls[0], Lsy = t.Ls[1], Lsz = t.Ls[2];
    const int kmax = A.kmax;
    for (int o = tid; o < M.n_own; o += blockDim.x) {
        int q, al;
        const int a = map_own(M, o, q, al);
        const float4 pi = sm[al];
        const int run = M.orun[q];
        const int hx = run % hn0, hy = (run / hn0) % hn1, hz = run / (hn0 * hn1);
        const int x0 = max(hx - 1, 0), x1 = min(hx + 1, hn0 - 1);
        uint2 *row = A.nl_tmp + tbsma_lrow(a, kmax >> 2);
        unsigned w0 = 0u, w1 = 0u;
        int cnt = 0, cnt_in = 0;
        for (int zz = max(hz - 1, 0); zz <= min(hz + 1, hn2 - 1); ++zz)
            for (int yy = max(hy - 1, 0); yy <= min(hy + 1, hn1 - 1); ++yy) {
                const int rb = (zz * hn1 + yy) * hn0;
                const int sb = M.lstart[rb + x0], e = M.lstart[rb + x1 + 1];
                for (int j = sb; j < e; ++j) {
                    const float4 pj = sm[j];
                    const float dx = wrap_d(pi.x - pj.x, hLx, Lsx), dy = wrap_d(pi.y - pj.y, hLy, Lsy);
                    const float dz = wrap_d(pi.z - pj.z, hLz, Lsz);
                    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));   // D:A6
                    if (d2 < A.ro2 && j != al) {
                        if (cnt < kmax) {
                            const unsigned v = (unsigned)j << ((cnt & 1) << 4);
                            if (cnt & 2) w1 |= v; else w0 |= v;
                            if ((cnt & 3) == 3) {
                                row[(size_t)(cnt >> 2) * TBSMA_LROW] = make_uint2(w0, w1);
                                w0 = w1 = 0u;
                            }
                        }
                        ++cnt;
                        cnt_in += d2 < A.rl2;
                    }
                }
            }
        if (cnt > kmax) atomicOr(A.ctrl + 1, (int)TBSMA_FLAG_NLIST_OVERFLOW);
        cnt = min(cnt, kmax);
        if (cnt & 3) row[(size_t)(cnt >> 2) * TBSMA_LROW] = make_uint2(w0, w1);
        cnts[o] = (unsigned short)cnt_in;
        A.nn_tmp[a] = cnt | ((__float_as_int(pi.w) & 3) << 16);
    }
    __syncthreads();
    for (int o = tid; o < M.n_own; o += blockDim.x) {
        int q, al;
        const int a = map_own(M, o, q, al);
        const int l0 = M.ostart[q], l1 = M.ostart[q + 1];
        const int my = cnts[o];
        int rank = 0;
        for (int b = l0; b < l1; ++b) {
            const int cb = cnts[b];
            rank += (cb > my) || (cb == my && b < o);
        }
        const int ns = M.gslot[M.orun[q]] + rank;
        A.newslot[a] = ns;
        A.oldof[ns] = a;
    }
}

// K1 over the tiles of the replicas whose candidates are rebuilt (work list 1)
__global__ void __launch_bounds__(kScanThreads)
k_tile_scan(const TileDesc *__restrict__ tiles, const int *__restrict__ work, int n_tiles, ScanArgs A)
{
    const int nw = work[1];
    for (int w = blockIdx.x; w < nw; w += gridDim.x) {
        __syncthreads();       // the previous tile's shared-memory image is no longer read
        const TileDesc t = tiles[work[2 + n_tiles + w]];
        if (t.kind == 0) scan_tile(t, A);
        else scan_box(t, A);
    }
}

// ---- K1b: placement of the halo records in the tile's shared-memory image.  The bank group ("class") a record is
// read from is its image index mod 8, and the gather passes read without bank conflicts only as far as every atom's
// neighbours are spread EVENLY over the eight classes (position p of lane l reads class (l + p) mod 8; a class that
// runs out leaves a hole that collides with a neighbour lane).  With the records simply in slot order the classes
// of an atom's ~70 neighbours are as good as random: 8.8 +- 2.8 per class, 7 holes per atom.  Here every atom gets a
// COLOUR from the cell of side h (default r0 / sqrt 2, the spacing of the (100) planes of the fcc lattice the
// potential describes) its position falls in, (ix + 2 iy + 3 iz) mod 8, and the image holds the records of colour c
// at indices 8 j + c + 1 (j = rank among the tile's records of that colour, in slot order; index 0 = sentinel).  On a
// crystal every sphere then holds nearly equal numbers of each colour (1 - 3 holes per atom); on a disordered
// system the colours are no worse than random.  Any placement is CORRECT: lists hold image offsets, whatever they are.
struct PlaceArgs {
    const int *cell_start, *oldof;
    const float4 *pos_sorted;        // cell-ordered positions of this rebuild
    const RepGeom *geom;
    unsigned short *img;             // per tile: halo-local index -> image index
    int *inv;                        // per tile: image index -> slot (inspection calls)
    int img_stride, inv_stride;      // tile_cap, img_cap
    int img_cap;                     // records an image may hold (sentinel included)
    float inv_h;                     // 1 / h; 0 = slot order (colour = index mod 8)
    int *ctrl;
};

__global__ void __launch_bounds__(256)
k_tile_place(const TileDesc *__restrict__ tiles, const int *__restrict__ work, int n_tiles, PlaceArgs A)
{
    __shared__ unsigned char s_col[TBSMA_TILE_MAX_RECORDS + 1];
    __shared__ int s_fallback;
    __shared__ TileMap M;
    const int nw = work[1];
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    for (int w = blockIdx.x; w < nw; w += gridDim.x) {
        const int ti = work[2 + n_tiles + w];
        const TileDesc t = tiles[ti];
        __syncthreads();
        tile_map_build(t, A.cell_start, M);
        struct { int nh; } r = {M.nh};
        if (M.n_own <= 0 || r.nh > A.img_stride) continue;
        const RepGeom *g = A.geom + t.rep;
        unsigned short *img = A.img + (size_t)ti * A.img_stride;
        int *inv = A.inv + (size_t)ti * A.inv_stride;
        __syncthreads();
        if (tid == 0) s_fallback = 0;
        for (int pass = 0; pass < 2; ++pass) {
            // pass 0: colours from the positions; pass 1 (only if they filled the image too unevenly): slot order
            for (int k = tid; k < r.nh; k += blockDim.x) {
                int col = k & 7;
                if (pass == 0 && A.inv_h > 0.f) {
                    const float4 p = A.pos_sorted[A.oldof[map_slot(M, k)]];
                    const int ix = __float2int_rd((p.x - g->lo[0]) * A.inv_h), iy = __float2int_rd((p.y - g->lo[1]) * A.inv_h);
                    const int iz = __float2int_rd((p.z - g->lo[2]) * A.inv_h);
                    col = (ix + 2 * iy + 3 * iz) & 7;
                }
                s_col[k] = (unsigned char)col;
            }
            __syncthreads();
            if (wid < 8) {         // warp c ranks the records of colour c in slot order
                int run = 0;
                for (int kb = 0; kb < r.nh; kb += 32) {
                    const int k = kb + lane;
                    const bool mine = k < r.nh && s_col[k] == wid;
                    const unsigned m = __ballot_sync(0xffffffffu, mine);
                    if (mine) {
                        const int idx = 8 * (run + __popc(m & ((1u << lane) - 1u))) + wid + 1;
                        if (idx < A.img_cap) { img[k] = (unsigned short)idx; inv[idx] = map_slot(M, k); }
                    }
                    run += __popc(m);
                }
                if (lane == 0 && 8 * (run - 1) + wid + 1 >= A.img_cap) s_fallback = 1;
            }
            __syncthreads();
            if (!s_fallback || pass == 1) break;
            __syncthreads();
        }
    }
}

__device__ __forceinline__ unsigned byte_of(unsigned long long v, int c) { return (unsigned)(v >> (c << 3)) & 0xffu; }

// ---- K2: finish.  One thread per FINAL slot of the tile: reads the temporary row of the atom that
// moves there, translates every partner to its final position (byte offset of its record in the
// tile's shared-memory image, 16 x the index k_tile_place gave it, the sentinel at 0), and writes the row sorted
// by CLASS (bank group of the record = record index mod 8; stable inside a class), starting with the
// class equal to the atom's lane mod 8: the inner build keeps this order when it filters, so its kept
// entries come out grouped by class as well, and while it gathers the candidates the eight lanes served by
// one shared-memory wavefront are (mostly) on eight different classes instead of all on class 0.
struct FinishArgs {
    const int *cell_start;
    const uint2 *nl_tmp;
    const int *nn_tmp, *newslot, *oldof;
    uint2 *nl;
    int *nn, *tileof;
    const unsigned short *img;   // image placement of every tile (k_tile_place)
    int img_stride;
    int n_pad, s_cap;
    int kg_o;                    // rows of capacity per atom of the candidate list (kmax_o / 4)
};

__device__ __forceinline__ void finish_tile(const TileDesc &t, int ti, const FinishArgs &A)
{
    const int *__restrict__ cell_start = A.cell_start;
    const uint2 *__restrict__ nl_tmp = A.nl_tmp;
    const int *__restrict__ nn_tmp = A.nn_tmp, *__restrict__ newslot = A.newslot;
    uint2 *__restrict__ nl = A.nl;
    int *__restrict__ nn = A.nn;
    const int s_cap = A.s_cap;
    extern __shared__ float4 smem_f4[];
    unsigned short *map = reinterpret_cast<unsigned short *>(smem_f4);   // s_cap entries
    __shared__ TileMap M;
    tile_map_build(t, cell_start, M);
    if (M.n_own <= 0 || M.nh > s_cap) return;
    const int tid = threadIdx.x;
    const unsigned short *__restrict__ img = A.img + (size_t)ti * A.img_stride;
    // cell-order halo-local index -> byte offset of the record in the image: the atom moves inside its run only
    for (int k = tid; k < M.nh; k += blockDim.x) {
        const int sc = map_slot(M, k);
        map[k] = (unsigned short)((unsigned)img[k + (newslot[sc] - sc)] << 4);
    }
    __syncthreads();
    // (thread per atom in CELL order, so that the reads of the temporary rows are coalesced; the atom's final slot ip, in
    // the same run, and with it its own-local index o there, follow from newslot)
    for (int oc = tid; oc < M.n_own; oc += blockDim.x) {
        int q, kh;
        const int a = map_own(M, oc, q, kh);
        const int ip = newslot[a];
        const int o = M.ostart[q] + (ip - M.gslot[M.orun[q]]);
        const int nnv = nn_tmp[a];
        const int cnt = nnv & 0xffff;
        const uint2 *src = nl_tmp + tbsma_lrow(a, A.kg_o);
        const int ng = (cnt + 3) >> 2;
        const unsigned lane = (unsigned)o & 31u;     // the lane the inner build and the gather passes give this atom
        // pass A: population of the 8 classes, counted from the lane's own (packed bytes; kmax <= 248)
        unsigned long long pop = 0ull;
        for (int g = 0; g < ng; ++g) {
            const uint2 w = src[(size_t)g * TBSMA_LROW];
            const unsigned e[4] = {w.x & 0xffffu, w.x >> 16, w.y & 0xffffu, w.y >> 16};
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (4 * g + q < cnt) pop += 1ull << ((((map[e[q]] >> 4) - lane) & 7) << 3);
        }
        unsigned long long off = 0ull;
        {
            unsigned run = 0;
#pragma unroll
            for (int c = 0; c < 8; ++c) { off |= (unsigned long long)run << (c << 3); run += byte_of(pop, c); }
        }
        // pass B: every entry straight to its class-sorted place in the atom's rows (two-byte stores that the L2 merges: a
        // shared-memory staging column per thread capped the CTA at 384 threads, one CTA per SM)
        unsigned short *dst16 = reinterpret_cast<unsigned short *>(nl + tbsma_lrow(ip, A.kg_o));
        unsigned long long cur = 0ull;
        for (int g = 0; g < ng; ++g) {
            const uint2 w = src[(size_t)g * TBSMA_LROW];
            const unsigned e[4] = {w.x & 0xffffu, w.x >> 16, w.y & 0xffffu, w.y >> 16};
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (4 * g + q < cnt) {
                    const unsigned m = map[e[q]];
                    const int c = ((m >> 4) - lane) & 7;
                    const unsigned idx = byte_of(off, c) + byte_of(cur, c);
                    cur += 1ull << (c << 3);
                    dst16[(size_t)(idx >> 2) * (TBSMA_LROW * 4) + (idx & 3u)] = (unsigned short)m;
                }
        }
        for (int k = cnt; k < 4 * ng; ++k)       // unused entries of the last row = 0 = the sentinel
            dst16[(size_t)(k >> 2) * (TBSMA_LROW * 4) + (k & 3)] = (unsigned short)0;
        nn[ip] = nnv;
        A.tileof[ip] = ti;
    }
}

__global__ void __launch_bounds__(kFinishMaxThreads)
k_tile_finish(const TileDesc *__restrict__ tiles, const int *__restrict__ work, int n_tiles, FinishArgs A)
{
    const int nw = work[1];
    for (int w = blockIdx.x; w < nw; w += gridDim.x) {
        __syncthreads();
        const int ti = work[2 + n_tiles + w];
        finish_tile(tiles[ti], ti, A);
    }
}

// ---- K3: move positions / velocities / tags from cell order to the final order and record the
// positions the candidates were built for.
__global__ void k_tile_permute(float4 *__restrict__ pos, float4 *__restrict__ vel, int *__restrict__ tag,
                               float4 *__restrict__ pos_outer, const int *__restrict__ atom_rep,
                               DirtyView dv, const int *__restrict__ oldof, const float4 *__restrict__ tmp_pos,
                               const float4 *__restrict__ tmp_vel, const int *__restrict__ tmp_tag, int n)
{
    if (!*dv.any) return;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        if (dv.dirty[atom_rep[k]] < dv.level) continue;
        const int a = oldof[k];
        const float4 p = tmp_pos[a];
        pos[k] = p;
        pos_outer[k] = p;
        if (vel) vel[k] = tmp_vel[a];
        tag[k] = tmp_tag[a];
    }
}

// API path of tbsma_build_neighbors: stage the caller's arrays as the "cell-ordered" source of K3
__global__ void k_stage_copy(const float4 *__restrict__ pos, const float4 *__restrict__ vel,
                             const int *__restrict__ tag, float4 *__restrict__ tmp_pos,
                             float4 *__restrict__ tmp_vel, int *__restrict__ tmp_tag, int n)
{
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        tmp_pos[k] = pos[k];
        if (vel) tmp_vel[k] = vel[k];
        tmp_tag[k] = tag[k];
    }
}

// ---- the two gather passes ---------------------------------------------------------------------
// Shared-memory image of a tile: record 0 is a sentinel far from everything (list rows are padded
// with offset 0 to a multiple of four entries: it fails the cutoff test like any distant atom, so
// the loops need no self / padding test), record k + 1 is the atom at slot halo_lo + k.
#define TBSMA_SENTINEL 1.0e9f

// The records of the halo go to the image indices k_tile_place chose for them (see there): one coalesced read of
// the slot range, scattered 16-byte stores.  The caller has made sure (__syncthreads) that nobody still reads a
// previous image.  (A contiguous image was one cp.async.bulk; spreading the records over the bank groups is worth
// more than the copy engine: a fifth fewer shared-memory wavefronts in the gather passes, 62 % fewer bank conflicts.)
__device__ __forceinline__ void fill_image(float4 *sm, const float4 *__restrict__ src,
                                           const unsigned short *__restrict__ img, const TileMap &M)
{
    const int nh = M.nh;
    if (threadIdx.x == 0) sm[0] = make_float4(TBSMA_SENTINEL, TBSMA_SENTINEL, TBSMA_SENTINEL, 0.f);
    if (!M.contig) {
        // box tile: run by run (a halo cell of ~60 records each), a warp per run, no search for the slot of a record
        const int lane = threadIdx.x & 31, nw = blockDim.x >> 5;
        for (int r = threadIdx.x >> 5; r < M.n_runs; r += nw) {
            const int s0 = M.lstart[r], e0 = M.lstart[r + 1], g0 = M.gslot[r] - s0;
            for (int k = s0 + lane; k < e0; k += 64) {
                const bool two = k + 32 < e0;
                const unsigned short a0 = img[k], a1 = two ? img[k + 32] : (unsigned short)0;
                const float4 r0 = src[g0 + k];
                float4 r1 = r0;
                if (two) r1 = src[g0 + k + 32];
                sm[a0] = r0;
                if (two) sm[a1] = r1;
            }
        }
        __syncthreads();
        return;
    }
    // eight records per thread and round, all sixteen loads in flight before the first store
    const int nthr = blockDim.x;
    for (int k0 = threadIdx.x; k0 < nh; k0 += 8 * nthr) {
        float4 rec[8];
        unsigned short at[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const int k = k0 + u * nthr;
            if (k < nh) { at[u] = img[k]; rec[u] = src[map_slot(M, k)]; }
        }
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (k0 + u * nthr < nh) sm[at[u]] = rec[u];
    }
    __syncthreads();
}

__device__ __forceinline__ float4 lds_rec(const float4 *sm, unsigned byte_off)
{
    return *reinterpret_cast<const float4 *>(reinterpret_cast<const char *>(sm) + byte_off);
}

// ---- packed fp32 arithmetic.  sm_100 has two-wide fp32 instructions (FADD2 / FMUL2 / FFMA2 on a pair of
// registers): the same flops per cycle as the scalar forms but half the issue slots, and both gather passes
// are bound by issue slots and the MUFU pipe, not by flops.  Two neighbours are evaluated side by side;
// every component sees exactly the operations of the scalar form (same roundings, D:A6 included).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpk(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
#define TBSMA_T_OUT 1.0e6f   // r - r0 of a pair outside the cutoff: every exponential of the pair becomes exactly 0

// d2 (D:A6 order), 1/r and t = r - r0 of two neighbours; t = TBSMA_T_OUT outside the cutoff
struct Pair2 {
    f32x2 dx, dy, dz, rinv, t;
};
// a tile whose halo wraps around periodic axes (TileDesc::Ls, hL): d += Ls where |d| > hL, which is D:A6's minimum image
// for every pair of an own atom and a staged record of that tile.  As m * Ls + d with m = 1.0 or 0.0: the product is
// exact, the sum rounds once, like the addition it stands for (and adding 0 changes nothing).
struct WrapC { float hLx, hLy, hLz, Lsx, Lsy, Lsz; };
__device__ __forceinline__ float set_gt_abs(float d, float h)
{
    float m;
    asm("set.gt.f32.f32 %0, %1, %2;" : "=f"(m) : "f"(fabsf(d)), "f"(h));
    return m;
}
template <bool WRAP>
__device__ __forceinline__ Pair2 pair2(const float4 &pi, const float4 &pa, const float4 &pb, const PairConst &pc,
                                       const WrapC &wc)
{
    Pair2 P;
    P.dx = pk(pi.x - pa.x, pi.x - pb.x);
    P.dy = pk(pi.y - pa.y, pi.y - pb.y);
    P.dz = pk(pi.z - pa.z, pi.z - pb.z);
    if (WRAP) {
        float a, b;
        unpk(P.dx, a, b); P.dx = fma2(pk(set_gt_abs(a, wc.hLx), set_gt_abs(b, wc.hLx)), pk(wc.Lsx, wc.Lsx), P.dx);
        unpk(P.dy, a, b); P.dy = fma2(pk(set_gt_abs(a, wc.hLy), set_gt_abs(b, wc.hLy)), pk(wc.Lsy, wc.Lsy), P.dy);
        unpk(P.dz, a, b); P.dz = fma2(pk(set_gt_abs(a, wc.hLz), set_gt_abs(b, wc.hLz)), pk(wc.Lsz, wc.Lsz), P.dz);
    }
    const f32x2 d2 = fma2(P.dz, P.dz, fma2(P.dy, P.dy, mul2(P.dx, P.dx)));
    float d2a, d2b;
    unpk(d2, d2a, d2b);
    P.rinv = pk(rsqrt_approx(d2a), rsqrt_approx(d2b));
    const f32x2 t = fma2(d2, P.rinv, pk(-pc.r0f, -pc.r0f));      // r - r0
    float ta, tb;
    unpk(t, ta, tb);
    P.t = pk(d2a < pc.rc2 ? ta : TBSMA_T_OUT, d2b < pc.rc2 ? tb : TBSMA_T_OUT);
    return P;
}

// xi^2 e^{-2q x} of two neighbours added to the two running sums in rho2
template <bool WRAP = false>
__device__ __forceinline__ f32x2 rho_term2(const float4 &pi, const float4 &pa, const float4 &pb, const PairConst &pc,
                                           f32x2 rho2, const WrapC &wc = WrapC())
{
    const Pair2 P = pair2<WRAP>(pi, pa, pb, pc, wc);
    const f32x2 arg = fma2(pk(pc.aq, pc.aq), P.t, pk(pc.b_rho, pc.b_rho));
    float a0, a1;
    unpk(arg, a0, a1);
    return add2(rho2, pk(ex2_approx(a0), ex2_approx(a1)));
}


// ---- inner build: the list the gather passes read, filtered from the candidates.
// Runs on the tile that owns the atoms, on the positions staged in shared memory (sm: record k + 1 =
// slot halo_lo + k, record 0 = sentinel).  The membership test is the fp32 predicate of D:A6 against
// rl2.  Also records the positions of this build (displacement check of the integrator) and compares
// them with those of the candidate build: more than S/2 away invalidates the candidates (status
// flag), more than want2^(1/2) asks for new candidates at the replica's next rebuild.
//
// Order of the kept entries (bank schedule).  A 128-bit shared-memory load is served eight lanes at a
// time, and eight lanes reading eight different 16-byte bank groups ("classes", record index mod 8) take
// one wavefront.  In the gather passes the atom is handled by lane l = (slot - first own slot) & 31 and
// all lanes are at the same list position p, so position p of lane l should hold a record of class
// (l + p) mod 8.  The candidates arrive sorted by class (K2), so the kept entries are eight runs, one per
// class; the list is written round by round, round j taking the j-th entry of the classes l, l + 1, ...,
// l + 7 (mod 8) that still have one.  While every class has a j-th entry that IS the schedule; when
// classes run out the later entries close up.
struct InnerArgs {
    const uint2 *olist;      // candidates (class-sorted rows)
    const int *nn_o;
    uint2 *nl;               // out: inner list            } both halves; the half NOT in use by the replica
    int *nn;                 // out: count | flag << 16    } is written (the last kernel of the step swaps)
    float4 *pos_build;       // out                        }
    const int *cur;          // per replica: half in use
    const unsigned short *img;   // image placement of every tile (k_tile_place)
    int img_stride, img_cap;
    size_t nl_stride;        // uint2 elements between the halves of nl
    int n_stride;            // elements between the halves of nn and pos_build
    const float4 *pos_outer;
    int *want_outer;         // per replica
    int kmax;                // inner capacity
    int kg_o;                // rows of capacity per atom of the candidate list
    float rl2, want2, viol2;
};

constexpr int kInnerThreads = 256;   // one atom per thread, kmax u16 of shared-memory scratch each

// tmp: element k of thread t at [k * nthr + t], kmax + 1 rows (row kmax takes what does not fit)
template <bool WRAP>
__device__ __forceinline__ void tile_inner_build(const TileDesc &t, const TileMap &M, int o_begin, int o_end,
                                                 const float4 *sm, const float4 *__restrict__ pos, unsigned short *tmp,
                                                 const InnerArgs &ia, int *__restrict__ ctrl)
{
    // o_begin is a multiple of 32, so tid & 31 is the lane the gather kernels give the atom
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31;
    int maxc = 0;
    bool want = false, viol = false, over = false;
    const int ob = ia.cur[t.rep] ^ 1;                  // the half to write
    uint2 *nl_out = ia.nl + (size_t)ob * ia.nl_stride;
    int *nn_out = ia.nn + (size_t)ob * ia.n_stride;
    float4 *pb_out = ia.pos_build + (size_t)ob * ia.n_stride;
    unsigned short *col = tmp + tid;
    for (int o = o_begin + tid; o < o_end; o += nthr) {
        const int i = map_own(M, o);
        const float4 pi = pos[i];
        const int nno = ia.nn_o[i];
        const int ng = ((nno & 0xffff) + 3) >> 2;
        const uint2 *row = ia.olist + tbsma_lrow(i, ia.kg_o);
        // pass 1: the candidates that pass the fp32 predicate of D:A6, in candidate order.  Branch-free: every
        // candidate is stored at the current end of the column, the end advances for the members only.
        int m = 0;
        auto group = [&](const uint2 jj) {
            const unsigned e[4] = {jj.x & 0xffffu, jj.x >> 16, jj.y & 0xffffu, jj.y >> 16};
            float d2[4];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const float4 pj = lds_rec(sm, e[q]);
                float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
                if (WRAP) { dx = wrap_d(dx, t.hL[0], t.Ls[0]); dy = wrap_d(dy, t.hL[1], t.Ls[1]); dz = wrap_d(dz, t.hL[2], t.Ls[2]); }
                d2[q] = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));   // D:A6
            }
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                col[min(m, ia.kmax) * nthr] = (unsigned short)e[q];
                m += d2[q] < ia.rl2 ? 1 : 0;       // padding entries point at the sentinel and fail
            }
        };
        {
            auto ld = [&](int g) { return g < ng ? __ldcs(row + (size_t)g * TBSMA_LROW) : make_uint2(0u, 0u); };
            uint2 q0 = ld(0), q1 = ld(1), q2 = ld(2), q3 = ld(3);
            int g = 0;
            for (; g + 4 <= ng; g += 4) {
                uint2 jj = q0; q0 = ld(g + 4); group(jj);
                jj = q1; q1 = ld(g + 5); group(jj);
                jj = q2; q2 = ld(g + 6); group(jj);
                jj = q3; q3 = ld(g + 7); group(jj);
            }
            if (g < ng) group(q0);
            if (g + 1 < ng) group(q1);
            if (g + 2 < ng) group(q2);
        }
        over = over || m > ia.kmax;
        maxc = max(maxc, m);
        m = min(m, ia.kmax);
        // entries per class, byte s = class lane + s (the order the classes are stored in), and where each run starts
        unsigned long long npk = 0ull;
        for (int k = 0; k < m; ++k) npk += 1ull << ((((col[k * nthr] >> 4) - (unsigned)lane) & 7u) << 3);
        unsigned long long orot = 0ull;
        int n_s[8];
        {
            unsigned run = 0;
#pragma unroll
            for (int sft = 0; sft < 8; ++sft) {
                n_s[sft] = (int)byte_of(npk, sft);
                orot |= (unsigned long long)run << (sft << 3);
                run += (unsigned)n_s[sft];
            }
        }
        // pass 2: position 8 j + s takes the j-th entry of class lane + s for j < L = m / 8.  A class with fewer than
        // L entries leaves holes; they, and the positions from 8 L on, take the entries beyond the L-th of the longer
        // classes, in stored order.
        uint2 *dst = nl_out + tbsma_lrow(i, ia.kmax >> 2);
        unsigned long long w = 0ull;
        const int L = m >> 3;
        int sc = 0, sj = L;
        auto next_surplus = [&]() {
            while (sj >= (int)byte_of(npk, sc)) { ++sc; sj = L; }
            return (int)byte_of(orot, sc) + sj++;
        };
        int o_s[8];
#pragma unroll
        for (int sft = 0; sft < 8; ++sft) o_s[sft] = (int)byte_of(orot, sft);
        for (int j = 0; j < L; ++j) {
#pragma unroll
            for (int sft = 0; sft < 8; ++sft) {
                const int k = n_s[sft] > j ? o_s[sft] + j : next_surplus();
                w |= (unsigned long long)col[k * nthr] << ((sft & 3) << 4);
                if ((sft & 3) == 3) {
                    dst[(size_t)(2 * j + (sft >> 2)) * TBSMA_LROW] = make_uint2((unsigned)w, (unsigned)(w >> 32));
                    w = 0ull;
                }
            }
        }
        for (int p = L << 3; p < m; ++p) {
            const int k = next_surplus();
            w |= (unsigned long long)col[k * nthr] << ((p & 3) << 4);
            if ((p & 3) == 3) {
                dst[(size_t)(p >> 2) * TBSMA_LROW] = make_uint2((unsigned)w, (unsigned)(w >> 32));
                w = 0ull;
            }
        }
        if (m & 3) dst[(size_t)(m >> 2) * TBSMA_LROW] = make_uint2((unsigned)w, (unsigned)(w >> 32));   // unused = 0 = sentinel
        nn_out[i] = m | (nno & 0x7fff0000);
        pb_out[i] = pi;
        const float4 po = ia.pos_outer[i];
        const float ox = pi.x - po.x, oy = pi.y - po.y, oz = pi.z - po.z;
        const float o2 = ox * ox + oy * oy + oz * oz;
        want = want || o2 > ia.want2;
        viol = viol || o2 > ia.viol2;
    }
    maxc = __reduce_max_sync(__activemask(), maxc);
    if (lane == 0 && maxc > 0) atomicMax(ctrl + 2, maxc);
    if (want) ia.want_outer[t.rep] = 1;
    if (viol) atomicOr(ctrl + 1, (int)TBSMA_FLAG_SKIN_VIOLATED);
    if (over) atomicOr(ctrl + 1, (int)TBSMA_FLAG_NLIST_OVERFLOW);
}

// inner build of the replicas on work list `which`, every tile cut into pieces of blockDim.x own atoms
__global__ void __launch_bounds__(kInnerThreads)
k_tile_inner(const TileDesc *__restrict__ tiles, const int *__restrict__ work, const int *__restrict__ cell_start,
             const float4 *__restrict__ pos, InnerArgs ia, int *__restrict__ ctrl, int n_pad, int s_cap, int nsplit,
             int which, int n_tiles)
{
    extern __shared__ float4 smem_f4[];
    __shared__ TileMap M;
    // the density pass may be launched as a programmatic dependent of this kernel (it reads the half of the list
    // buffers this kernel does not write): let it start at once
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    const int *__restrict__ wl = work + 2 + which * n_tiles;
    const int nu = work[which] * nsplit;
    if ((int)blockIdx.x >= nu) return;
    unsigned short *tmp = reinterpret_cast<unsigned short *>(smem_f4 + ia.img_cap);
    for (int u = blockIdx.x; u < nu; u += gridDim.x) {
        const int ti = wl[u / nsplit];
        const TileDesc t = tiles[ti];
        __syncthreads();       // nobody still reads the previous map or image
        tile_map_build(t, cell_start, M);
        const int o_begin = (u % nsplit) * blockDim.x;
        if (o_begin >= M.n_own) continue;
        if (M.nh > s_cap) {
            if (threadIdx.x == 0) atomicOr(ctrl + 1, (int)TBSMA_FLAG_TILE_OVERFLOW);
            continue;
        }
        fill_image(smem_f4, pos, ia.img + (size_t)ti * ia.img_stride, M);
        // the last piece also takes whatever a tile holds beyond the headroom it was sized with
        const int o_end = (u % nsplit) == nsplit - 1 ? M.n_own : min(o_begin + (int)blockDim.x, M.n_own);
        if (t.Ls[0] != 0.f || t.Ls[1] != 0.f || t.Ls[2] != 0.f) tile_inner_build<true>(t, M, o_begin, o_end, smem_f4, pos, tmp, ia, ctrl);
        else tile_inner_build<false>(t, M, o_begin, o_end, smem_f4, pos, tmp, ia, ctrl);
    }
}

// Work distribution of the two gather kernels: the own atoms of a tile are cut into chunks of 32
// consecutive slots (equal list lengths, thanks to the count order) and the warps of the CTA take
// chunks from a shared counter, so no warp waits at the end for one that drew the long lists.
// The list rows are prefetched three groups (12 entries) ahead: a row is 8 bytes per lane from
// HBM, and one group of pair terms is shorter than the HBM latency.
__device__ __forceinline__ int next_chunk(int *counter)
{
    int ch = 0;
    if ((threadIdx.x & 31) == 0) ch = atomicAdd(counter, 1);
    return __shfl_sync(0xffffffffu, ch, 0);
}

__device__ __forceinline__ uint2 ld_row(const uint2 *row, int g, int ng, int n_pad)
{
    return g < ng ? __ldcs(row + (size_t)g * TBSMA_LROW) : make_uint2(0u, 0u);
}

// stage 1 (Eq.1): rho_i over the list, s_i = rho_i^(-1/2) packed with the position.
// SPLIT: the CTA takes part `part` of `nsplit` of the tile's chunks (small batches); otherwise all of them
template <bool SPLIT, bool WRAP>
__device__ __forceinline__ void density_tile(const TileDesc &t, const TileMap &M,
                                             const float4 *__restrict__ pos, const uint2 *__restrict__ nl,
                                             const int *__restrict__ nn, float4 *__restrict__ xs,
                                             int *__restrict__ ctrl, int n_pad, int s_cap, const PairConst &pc,
                                             const unsigned short *__restrict__ img, int part, int nsplit, int kg)
{
    struct { int lo, hi, nh; } r = {0, M.n_own, M.nh};      // own-local range
    if (r.hi <= r.lo) return;
    if (r.nh > s_cap) {
        if (threadIdx.x == 0) atomicOr(ctrl + 1, (int)TBSMA_FLAG_TILE_OVERFLOW);
        return;
    }
    const WrapC wc = {t.hL[0], t.hL[1], t.hL[2], t.Ls[0], t.Ls[1], t.Ls[2]};
    // this CTA's share of the tile's 32-atom chunks (all of them unless the batch is too small to fill the GPU)
    // (the range lives in shared memory: the loops below have no register to spare)
    extern __shared__ float4 smem_f4[];
    __shared__ int s_next, s_end;
    {
        const int nchunk_all = (r.hi - r.lo + 31) >> 5;
        const int cb = SPLIT ? nchunk_all * part / nsplit : 0, ce = SPLIT ? nchunk_all * (part + 1) / nsplit : nchunk_all;
        if (ce <= cb) return;
        if (threadIdx.x == 0) { s_next = cb; s_end = ce; }
    }
    const float4 *sm = smem_f4;
    fill_image(smem_f4, pos, img, M);
    const int lane = threadIdx.x & 31;
    const int nchunk = (r.hi - r.lo + 31) >> 5;
    for (int ch = next_chunk(&s_next); ch < (SPLIT ? s_end : nchunk); ch = next_chunk(&s_next)) {
        const int o = (ch << 5) + lane;
        if (o >= r.hi) continue;
        const int i = map_own(M, o);
        // own record, count and the first three rows in one round trip (the rows exist whatever the count: kg >= 3 or the
        // loads are skipped); a row register is reloaded right after its use
        const uint2 *row = nl + tbsma_lrow(i, kg);
        uint2 q0 = make_uint2(0u, 0u), q1 = q0, q2 = q0;
        if (kg >= 3) { q0 = __ldcs(row); q1 = __ldcs(row + TBSMA_LROW); q2 = __ldcs(row + 2 * TBSMA_LROW); }
        const float4 pi = pos[i];
        const int ng = ((nn[i] & 0xffff) + 3) >> 2;
        if (kg < 3) { q0 = ld_row(row, 0, ng, n_pad); q1 = ld_row(row, 1, ng, n_pad); q2 = ld_row(row, 2, ng, n_pad); }
        if (ng < 3) { q2 = make_uint2(0u, 0u); if (ng < 2) q1 = q2; if (ng < 1) q0 = q2; }
        f32x2 rho2 = pk(0.f, 0.f);
        auto group = [&](const uint2 jj) {
            const float4 p0 = lds_rec(sm, jj.x & 0xffffu), p1 = lds_rec(sm, jj.x >> 16);
            const float4 p2 = lds_rec(sm, jj.y & 0xffffu), p3 = lds_rec(sm, jj.y >> 16);
            rho2 = rho_term2<WRAP>(pi, p0, p1, pc, rho2, wc);
            rho2 = rho_term2<WRAP>(pi, p2, p3, pc, rho2, wc);
        };
        int g = 0;
        for (; g + 3 <= ng; g += 3) {
            group(q0); q0 = ld_row(row, g + 3, ng, n_pad);
            group(q1); q1 = ld_row(row, g + 4, ng, n_pad);
            group(q2); q2 = ld_row(row, g + 5, ng, n_pad);
        }
        if (g < ng) {
            group(q0);
            if (g + 1 < ng) group(q1);
        }
        float rho0, rho1;
        unpk(rho2, rho0, rho1);
        const float rho = rho0 + rho1;
        const float s = rho > 0.f ? 1.0f / sqrtf(rho) : 0.f;     // once per atom, IEEE (D:A5 for rho = 0)
        xs[i] = make_float4(pi.x, pi.y, pi.z, s);
    }
}

// Which half of the list buffers a tile reads: the one its replica has in use, or, when the replica's list has
// just been rebuilt ahead of this launch (dirty >= sync_level), the other one (the step's last kernel swaps).
struct ListSel {
    const int *cur, *dirty;
    int sync_level;          // 1: every rebuild of this step precedes the gather passes; 2: only those with new candidates
    size_t nl_stride;
    int n_stride;
    const unsigned short *img;   // image placement of every tile (k_tile_place)
    int img_stride;
    int nsplit;                  // CTAs per tile (> 1 when the tiles are too few to fill the GPU)
    int kg;                      // rows of capacity per atom of the list (kmax / 4)
};
__device__ __forceinline__ int list_half(const ListSel &ls, int rep)
{
    return ls.cur[rep] ^ (ls.dirty[rep] >= ls.sync_level ? 1 : 0);
}

// one CTA per tile (or per part of a tile, ls.nsplit).  nn and nl are read-only here: they were written by an earlier kernel (or, the half not read,
// are being written by the filter pass running beside this launch).
template <bool SPLIT>
__global__ void __launch_bounds__(512, 2)
k_density_tile(const TileDesc *__restrict__ tiles, const int *__restrict__ cell_start,
               const float4 *__restrict__ pos, const uint2 *__restrict__ nl, const int *__restrict__ nn,
               float4 *__restrict__ xs, int *__restrict__ ctrl, ListSel ls, int n_pad, int s_cap, PairConst pc)
{
    const int ti = SPLIT ? (int)blockIdx.x / ls.nsplit : (int)blockIdx.x, part = SPLIT ? (int)blockIdx.x % ls.nsplit : 0;
    const TileDesc t = tiles[ti];
    const int h = list_half(ls, t.rep);
    __shared__ TileMap M;
    tile_map_build(t, cell_start, M);
    if (t.Ls[0] != 0.f || t.Ls[1] != 0.f || t.Ls[2] != 0.f)
        density_tile<SPLIT, true>(t, M, pos, nl + (size_t)h * ls.nl_stride, nn + (size_t)h * ls.n_stride, xs, ctrl, n_pad,
                                  s_cap, pc, ls.img + (size_t)ti * ls.img_stride, part, ls.nsplit, ls.kg);
    else
        density_tile<SPLIT, false>(t, M, pos, nl + (size_t)h * ls.nl_stride, nn + (size_t)h * ls.n_stride, xs, ctrl, n_pad,
                                   s_cap, pc, ls.img + (size_t)ti * ls.img_stride, part, ls.nsplit, ls.kg);
    // Launched as a programmatic dependent of the filter kernel this pass starts early and reads nothing of it; but the
    // kernels after it (force pass, then the swap of the list halves) are ordered after THIS kernel only, so it must
    // not complete before the filter kernel has (a no-op for an ordinary launch).
    asm volatile("griddepcontrol.wait;" ::: "memory");
}

// running sums of stage 2, two lanes each (even / odd neighbours), added up once per atom
struct AccT {
    f32x2 fx, fy, fz, er;
    f32x2 wxx, wyy, wzz, wxy, wxz, wyz;
};

// Two neighbours of atom i (pi.w = s_i, pa.w / pb.w = s_j):
//   F_i += [ (2Ap/r0) e^{-p x} - (q xi^2/r0) e^{-2q x} (s_i + s_j) ] d_ij / r_ij   (derivative of Eq.1-3)
// and the repulsive sum of Eq.2.  Outside the cutoff t = TBSMA_T_OUT makes both exponentials exactly 0.
template <bool VIRIAL, bool WRAP = false>
__device__ __forceinline__ void force_term2(const float4 &pi, const float4 &pa, const float4 &pb, const PairConst &pc,
                                            AccT &a, const WrapC &wc = WrapC())
{
    const Pair2 P = pair2<WRAP>(pi, pa, pb, pc, wc);
    const f32x2 ar = fma2(pk(pc.ap, pc.ap), P.t, pk(pc.b_rep, pc.b_rep));
    const f32x2 ab = fma2(pk(pc.aq, pc.aq), P.t, pk(pc.b_band, pc.b_band));
    float ar0, ar1, ab0, ab1;
    unpk(ar, ar0, ar1);
    unpk(ab, ab0, ab1);
    const f32x2 er = pk(ex2_approx(ar0), ex2_approx(ar1));          // (2Ap/r0) e^{-p x}
    const f32x2 eb = pk(ex2_approx(ab0), ex2_approx(ab1));          // (q xi^2/r0) e^{-2q x}
    const f32x2 nss = pk(-pi.w - pa.w, -pi.w - pb.w);               // -(s_i + s_j)
    const f32x2 fp = mul2(fma2(eb, nss, er), P.rinv);               // -dE/dr / r
    a.fx = fma2(fp, P.dx, a.fx);
    a.fy = fma2(fp, P.dy, a.fy);
    a.fz = fma2(fp, P.dz, a.fz);
    a.er = add2(a.er, er);
    if (VIRIAL) {
        const f32x2 fx = mul2(fp, P.dx), fy = mul2(fp, P.dy), fz = mul2(fp, P.dz);
        a.wxx = fma2(P.dx, fx, a.wxx); a.wyy = fma2(P.dy, fy, a.wyy); a.wzz = fma2(P.dz, fz, a.wzz);
        a.wxy = fma2(P.dx, fy, a.wxy); a.wxz = fma2(P.dx, fz, a.wxz); a.wyz = fma2(P.dy, fz, a.wyz);
    }
}
__device__ __forceinline__ float sum2(f32x2 v)
{
    float lo, hi;
    unpk(v, lo, hi);
    return lo + hi;
}

__device__ __forceinline__ double warp_sum_d(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// a6.  Per-replica sums are ORDER-FIXED, so that energies, virials and kinetic energies are bitwise repeatable: the 32
// atoms of a chunk are added by a shuffle tree, the chunks of a CTA in chunk order (whichever warp happened to work on
// them), and tbsma_reduce_replicas (tbsma_internal.cuh) adds the CTAs of a replica in tile order.  No atomics.
constexpr int kMaxChunks = (TBSMA_TILE_MAX_RECORDS + 31) / 32 + 1;

// stage 2 (Eq.1-3, Eq.5): forces, per-atom energy, virial, closing half kick, E_kin
template <bool VIRIAL, bool KICK, bool SPLIT, bool WRAP>
__device__ __forceinline__ void force_tile(const TileDesc &t, const TileMap &M,
                                           const float4 *__restrict__ xs, const uint2 *__restrict__ nl,
                                           const int *__restrict__ nn, float4 *__restrict__ force, const KickArgs &kk,
                                           int *__restrict__ ctrl, int n_pad, int s_cap, const PairConst &pc,
                                           const unsigned short *__restrict__ img, int part, int nsplit,
                                           double *__restrict__ my_sums, int kg)
{
    constexpr int NQ = VIRIAL ? 8 : 2;
    __shared__ double s_part[NQ][kMaxChunks];
    const int lane = threadIdx.x & 31;
    // every CTA leaves its sums (E, E_kin, W): zero if it has nothing to do
    if (threadIdx.x < NQ) my_sums[threadIdx.x] = 0.0;
    struct { int lo, hi, nh; } r = {0, M.n_own, M.nh};      // own-local range
    const WrapC wc = {t.hL[0], t.hL[1], t.hL[2], t.Ls[0], t.Ls[1], t.Ls[2]};
    if (r.hi <= r.lo) return;
    if (r.nh > s_cap) {
        if (threadIdx.x == 0) atomicOr(ctrl + 1, (int)TBSMA_FLAG_TILE_OVERFLOW);
        return;
    }
    extern __shared__ float4 smem_f4[];
    __shared__ int s_next, s_end, s_begin;
    {
        const int nchunk_all = (r.hi - r.lo + 31) >> 5;
        const int cb = SPLIT ? nchunk_all * part / nsplit : 0, ce = SPLIT ? nchunk_all * (part + 1) / nsplit : nchunk_all;
        if (ce <= cb) return;
        if (threadIdx.x == 0) { s_next = cb; s_end = ce; s_begin = cb; }
    }
    const float4 *sm = smem_f4;
    fill_image(smem_f4, xs, img, M);
    bool bad = false;
    for (int ch = next_chunk(&s_next); ch < s_end; ch = next_chunk(&s_next)) {
        const int o = (ch << 5) + lane;
        double se = 0.0, sk = 0.0, sw[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
        if (o < r.hi) {
        const int i = map_own(M, o);
        const uint2 *row = nl + tbsma_lrow(i, kg);
        uint2 q0 = make_uint2(0u, 0u), q1 = q0, q2 = q0;
        if (kg >= 3) { q0 = __ldcs(row); q1 = __ldcs(row + TBSMA_LROW); q2 = __ldcs(row + 2 * TBSMA_LROW); }
        const float4 pi = xs[i];
        const int nni = nn[i];
        const int ng = ((nni & 0xffff) + 3) >> 2;
        if (kg < 3) { q0 = ld_row(row, 0, ng, n_pad); q1 = ld_row(row, 1, ng, n_pad); q2 = ld_row(row, 2, ng, n_pad); }
        if (ng < 3) { q2 = make_uint2(0u, 0u); if (ng < 2) q1 = q2; if (ng < 1) q0 = q2; }
        const f32x2 z2 = pk(0.f, 0.f);
        AccT a = {z2, z2, z2, z2, z2, z2, z2, z2, z2, z2};
        auto group = [&](const uint2 jj) {
            const float4 p0 = lds_rec(sm, jj.x & 0xffffu), p1 = lds_rec(sm, jj.x >> 16);
            const float4 p2 = lds_rec(sm, jj.y & 0xffffu), p3 = lds_rec(sm, jj.y >> 16);
            force_term2<VIRIAL, WRAP>(pi, p0, p1, pc, a, wc);
            force_term2<VIRIAL, WRAP>(pi, p2, p3, pc, a, wc);
        };
        int g = 0;
        for (; g + 3 <= ng; g += 3) {
            group(q0); q0 = ld_row(row, g + 3, ng, n_pad);
            group(q1); q1 = ld_row(row, g + 4, ng, n_pad);
            group(q2); q2 = ld_row(row, g + 5, ng, n_pad);
        }
        if (g < ng) {
            group(q0);
            if (g + 1 < ng) group(q1);
        }
        const float fx = sum2(a.fx), fy = sum2(a.fy), fz = sum2(a.fz);
        const float sqrt_rho = pi.w > 0.f ? 1.0f / pi.w : 0.f;
        const float ei = __fmaf_rn(sum2(a.er), pc.e_rep_scale, -sqrt_rho);   // Eq.1-3: E_R^i + E_B^i
        force[i] = make_float4(fx, fy, fz, ei);
        bad = bad || !isfinite(fx + fy + fz + ei);
        se = (double)ei;
        if (KICK && (nni >> 16) == 0) {       // final B of the step, dynamic atoms only
            float4 v = kk.vel[i];
            v.x = __fmaf_rn(kk.kick, fx, v.x);
            v.y = __fmaf_rn(kk.kick, fy, v.y);
            v.z = __fmaf_rn(kk.kick, fz, v.z);
            kk.vel[i] = v;
            sk = (double)(kk.ke_scale * (v.x * v.x + v.y * v.y + v.z * v.z));
        }
        if (VIRIAL) {
            sw[0] = 0.5 * (double)sum2(a.wxx); sw[1] = 0.5 * (double)sum2(a.wyy); sw[2] = 0.5 * (double)sum2(a.wzz);
            sw[3] = 0.5 * (double)sum2(a.wxy); sw[4] = 0.5 * (double)sum2(a.wxz); sw[5] = 0.5 * (double)sum2(a.wyz);
        }
        }
        // the chunk's sums, by a fixed tree
        __syncwarp();
        se = warp_sum_d(se);
        if (KICK) sk = warp_sum_d(sk);
        if (VIRIAL) {
#pragma unroll
            for (int k = 0; k < 6; ++k) sw[k] = warp_sum_d(sw[k]);
        }
        if (lane == 0) {
            const int c = ch - s_begin;
            s_part[0][c] = se;
            s_part[1][c] = sk;
            if (VIRIAL) {
#pragma unroll
                for (int k = 0; k < 6; ++k) s_part[(2 + k) % NQ][c] = sw[k];
            }
        }
    }
    if (bad) atomicOr(ctrl + 1, (int)TBSMA_FLAG_NONFINITE);
    __syncthreads();
    // the CTA's sums: chunks in chunk order (lane l takes chunks l, l + 32, ...; then a fixed tree)
    if (threadIdx.x < 32) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            double v = 0.0;
            for (int c = lane; c < s_end - s_begin; c += 32) v += s_part[q][c];
            v = warp_sum_d(v);
            if (lane == 0) my_sums[q] = v;
        }
    }
}

template <bool VIRIAL, bool KICK, bool SPLIT>
__global__ void __launch_bounds__(512, 2)
k_force_tile(const TileDesc *__restrict__ tiles, const int *__restrict__ cell_start,
             const float4 *__restrict__ xs, const uint2 *__restrict__ nl, const int *__restrict__ nn,
             float4 *__restrict__ force, double *__restrict__ cta_sums, KickArgs kk,
             int *__restrict__ ctrl, ListSel ls, int n_pad, int s_cap, PairConst pc)
{
    const int ti = SPLIT ? (int)blockIdx.x / ls.nsplit : (int)blockIdx.x, part = SPLIT ? (int)blockIdx.x % ls.nsplit : 0;
    const TileDesc t = tiles[ti];
    const int h = list_half(ls, t.rep);
    __shared__ TileMap M;
    tile_map_build(t, cell_start, M);
    if (t.Ls[0] != 0.f || t.Ls[1] != 0.f || t.Ls[2] != 0.f)
        force_tile<VIRIAL, KICK, SPLIT, true>(t, M, xs, nl + (size_t)h * ls.nl_stride, nn + (size_t)h * ls.n_stride, force,
                                              kk, ctrl, n_pad, s_cap, pc, ls.img + (size_t)ti * ls.img_stride, part,
                                              ls.nsplit, cta_sums + 8 * (size_t)blockIdx.x, ls.kg);
    else
        force_tile<VIRIAL, KICK, SPLIT, false>(t, M, xs, nl + (size_t)h * ls.nl_stride, nn + (size_t)h * ls.n_stride, force,
                                               kk, ctrl, n_pad, s_cap, pc, ls.img + (size_t)ti * ls.img_stride, part,
                                               ls.nsplit, cta_sums + 8 * (size_t)blockIdx.x, ls.kg);
}

// ---- the whole step of a small batch in ONE kernel ---------------------------------------
// The paper pays "+35 % run time due to thread synchronization" between its two stages; a single wire per GPU is its
// unit of work.  For a batch whose tiles (or parts of tiles) all fit the GPU at once the step is one cooperative
// launch: every CTA integrates its share of the atoms (B A O A, grips, displacement check), the grid synchronises, the CTA
// works its tile's chunks through the density pass, the grid synchronises, the force pass with the closing kick, the grid
// synchronises, and the first CTAs add up the replicas and do the step's bookkeeping.  Three grid barriers of about a
// microsecond in place of five kernel boundaries.  If the displacement check finds a replica that needs a new list the
// kernel stops after the integration and sets the graph conditional: the rest of that step (list renewal, density,
// force, bookkeeping) is run by the ordinary kernels in the body of an IF node.  Same device functions as the separate
// kernels, same order of operations: bit-identical results.
struct FusedArgs {
    // integration
    float4 *pos, *vel;
    float4 *force;
    const float4 *pos_build;
    const int *atom_rep;
    const RepGeom *geom;
    const int *tag;
    StepArgs a;
    unsigned long long *counters;
    int *dirty, *ctrl;
    int n, R;
    // gather passes
    const TileDesc *tiles;
    const int *cell_start;
    const uint2 *nl;
    const int *nn;
    float4 *xs;
    double *cta_sums;
    KickArgs kk;
    ListSel ls;
    int n_pad, s_cap;
    PairConst pc;
    // bookkeeping
    float *stagger;
    int *cur;
    int swap, advance, count_step;
    TileSums ts;
    cudaGraphConditionalHandle cond;
};

template <bool VIRIAL, bool SPLIT>
__global__ void __launch_bounds__(256, 4)
k_step_small(const FusedArgs F)
{
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    const int nthr = (int)(gridDim.x * blockDim.x);
    const int work = F.n > F.R ? F.n : F.R;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < work; i += nthr)
        tbsma_integrate_one(i, F.pos, F.vel, F.force, F.pos_build, F.atom_rep, F.geom, F.tag, F.a, F.counters, F.dirty, F.ctrl,
                            F.n, F.R);
    grid.sync();
    const int any_dirty = *(volatile int *)F.ctrl;
    if (blockIdx.x == 0 && threadIdx.x == 0) cudaGraphSetConditional(F.cond, any_dirty ? 1u : 0u);
    if (any_dirty) return;         // every CTA sees the same flag: nobody is left waiting at a barrier
    const int ti = SPLIT ? (int)blockIdx.x / F.ls.nsplit : (int)blockIdx.x, part = SPLIT ? (int)blockIdx.x % F.ls.nsplit : 0;
    const TileDesc t = F.tiles[ti];
    const int h = F.ls.cur[t.rep];
    const uint2 *nl = F.nl + (size_t)h * F.ls.nl_stride;
    const int *nn = F.nn + (size_t)h * F.ls.n_stride;
    const unsigned short *img = F.ls.img + (size_t)ti * F.ls.img_stride;
    __shared__ TileMap M;
    tile_map_build(t, F.cell_start, M);
    const bool wrap = t.Ls[0] != 0.f || t.Ls[1] != 0.f || t.Ls[2] != 0.f;
    if (wrap) density_tile<SPLIT, true>(t, M, F.pos, nl, nn, F.xs, F.ctrl, F.n_pad, F.s_cap, F.pc, img, part, F.ls.nsplit, F.ls.kg);
    else density_tile<SPLIT, false>(t, M, F.pos, nl, nn, F.xs, F.ctrl, F.n_pad, F.s_cap, F.pc, img, part, F.ls.nsplit, F.ls.kg);
    grid.sync();
    double *my_sums = F.cta_sums + 8 * (size_t)blockIdx.x;
    if (wrap) force_tile<VIRIAL, true, SPLIT, true>(t, M, F.xs, nl, nn, F.force, F.kk, F.ctrl, F.n_pad, F.s_cap, F.pc, img, part,
                                                    F.ls.nsplit, my_sums, F.ls.kg);
    else force_tile<VIRIAL, true, SPLIT, false>(t, M, F.xs, nl, nn, F.force, F.kk, F.ctrl, F.n_pad, F.s_cap, F.pc, img, part,
                                                F.ls.nsplit, my_sums, F.ls.kg);
    grid.sync();
    tbsma_reduce_replicas(F.ts, F.R);
    if (blockIdx.x == 0) tbsma_finish_bookkeeping(F.dirty, F.ctrl, F.stagger, F.cur, F.swap, F.counters, F.R, F.advance, F.count_step);
}

// ---- persistent gather kernels ----------------------------------------------------------------------
// One CTA of 16 warps per half SM for the whole pass.  Work comes in UNITS (a tile, or 1 / S of a tile's 32-atom chunks for
// the last tiles of the pass and for batches with few tiles), claimed from a global counter.  A CTA holds TWO tile images:
// while its warps work through the chunks of unit k the image of unit k + 1 is already in shared memory, and a warp that
// finds no chunk left in unit k moves on to unit k + 1 AT ONCE -- no CTA-wide barrier at the end of a tile (8 % of the
// warp time of the one-CTA-per-tile kernels: 25 chunks over 8 warps), no wait for an image fill (5 %), no partial last wave
// of CTAs (6 %).  The last warp out of unit k adds the unit's sums in chunk order, claims unit k + 2 and fills the image
// buffer unit k just vacated with cp.async (16 bytes per record, straight to the placed image index), completion
// signalled on an mbarrier the warps wait on before they enter unit k + 2.
struct PSlot {
    int tile;            // < 0: the pass has run out of units
    int lo, hi;          // own slots of the tile
    int cb, ce;          // chunks [cb, ce) of the tile are this unit's
    int half;            // which half of the list buffers the tile's replica reads
    int sums;            // slot in cta_sums (force pass)
    int pad;
};
constexpr int kPMaxBuf = 4;
struct PShared {
    unsigned long long full[kPMaxBuf];   // mbarriers: image + slot description of the buffer are in place
    PSlot slot[kPMaxBuf];
    int next[kPMaxBuf], done[kPMaxBuf];
    // the unit that comes to a buffer next, claimed and described by the FIRST warp that leaves the current one (the chain
    // claim -> tile -> cell_start -> list half is three dependent round trips to memory, off the filling warp's path)
    PSlot pend[kPMaxBuf];
    int pend_tile[kPMaxBuf], pend_hlo[kPMaxBuf], pend_nh[kPMaxBuf];
    volatile int pend_ok[kPMaxBuf];
    int ended;
};
constexpr int kPThreads = 512;
constexpr int kPWarps = kPThreads / 32;

struct PUnits {
    int n_units;     // n_plain whole tiles, then (n_tiles - n_plain) tiles in S parts each
    int n_plain, S;
    int max_chunks;  // capacity of the per-chunk sums of a unit
};
__device__ __forceinline__ void punit(const PUnits &U, int u, int &tile, int &part, int &nparts)
{
    if (u < U.n_plain) { tile = u; part = 0; nparts = 1; }
    else { const int v = u - U.n_plain; tile = U.n_plain + v / U.S; part = v % U.S; nparts = U.S; }
}

__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long *b, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long *b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long *b, unsigned parity)
{
    const unsigned a = smem_u32(b);
    unsigned ok;
    do {
        // (may suspend the thread for up to the hinted time instead of spinning through the issue slots)
        asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3; selp.u32 %0, 1, 0, p; }"
                     : "=r"(ok) : "r"(a), "r"(parity), "r"(2000u) : "memory");
    } while (!ok);
}

// description of unit u in slot b (lane 0 of the calling warp writes it); returns halo_lo and nh for the fill
__device__ __forceinline__ bool pslot_describe(PSlot &S, const PUnits &U, int u, const TileDesc *__restrict__ tiles,
                                               const int *__restrict__ cell_start, const ListSel &ls, int s_cap,
                                               int *__restrict__ ctrl, int &tile, int &halo_lo, int &nh)
{
    int part, nparts;
    punit(U, u, tile, part, nparts);
    const TileDesc t = tiles[tile];
    const TileRange r = tile_range(t, cell_start);
    S.tile = tile;
    S.lo = r.lo; S.hi = r.hi;
    S.half = list_half(ls, t.rep);
    S.sums = tile * U.S + part;
    const int nchunk_all = (r.hi - r.lo + 31) >> 5;
    S.cb = nchunk_all * part / nparts;
    S.ce = nchunk_all * (part + 1) / nparts;
    halo_lo = r.halo_lo; nh = r.nh;
    bool ok = r.hi > r.lo && S.ce > S.cb;
    if (r.nh > s_cap || S.ce - S.cb > U.max_chunks) {
        atomicOr(ctrl + 1, (int)TBSMA_FLAG_TILE_OVERFLOW);
        ok = false;
    }
    if (!ok) S.ce = S.cb;     // nothing to do (its sums are still written: zero)
    return ok;
}

// image fill by ONE warp, asynchronous: every lane's copies arrive on `bar` when they have landed
__device__ __forceinline__ void fill_image_async(float4 *sm, const float4 *__restrict__ src,
                                                 const unsigned short *__restrict__ img, int halo_lo, int nh,
                                                 unsigned long long *bar)
{
    const int lane = threadIdx.x & 31;
    const unsigned base = smem_u32(sm);
    // 32 image indices per lane in flight before the first copy is issued: two rounds for a tile of 2000 records
    for (int k0 = lane; k0 < nh; k0 += 32 * 32) {
        unsigned at[32];
#pragma unroll
        for (int u = 0; u < 32; ++u) at[u] = k0 + u * 32 < nh ? (unsigned)img[k0 + u * 32] : 0u;
#pragma unroll
        for (int u = 0; u < 32; ++u)
            if (k0 + u * 32 < nh)
                asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(base + (at[u] << 4)),
                             "l"(src + halo_lo + k0 + u * 32) : "memory");
    }
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// PASS 0: density (src = pos, out = xs); PASS 1: force (src = xs, out = force, sums, kick)
struct PArgs {
    const TileDesc *tiles;
    const int *cell_start;
    const float4 *src;
    const uint2 *nl;
    const int *nn;
    float4 *xs;            // density: out
    float4 *force;         // force: out
    double *cta_sums;      // force: out
    KickArgs kk;
    int *ctrl;
    int *claim;            // this pass's unit counter
    int *claim_other;      // the other pass's, reset here (the two passes never run together); both are also zeroed ahead
                           // of the density pass: by k_tile_worklist inside a step, by a memset node otherwise
    ListSel ls;
    int n_pad, s_cap, img_cap;
    int nb;                // image buffers per CTA (2 .. kPMaxBuf)
    PUnits U;
    PairConst pc;
};

template <int PASS, bool VIRIAL, bool KICK>
__global__ void __launch_bounds__(kPThreads, 2)
k_gather_persist(const PArgs A)
{
    constexpr int NQ = VIRIAL ? 8 : 2;
    extern __shared__ float4 smem_f4[];
    __shared__ PShared sh;
    const int NB = A.nb;
    double *s_part = reinterpret_cast<double *>(smem_f4 + (size_t)NB * A.img_cap);    // force: [NB][NQ][max_chunks]
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const int G = (int)gridDim.x;
    if (blockIdx.x == 0 && threadIdx.x == 0) *A.claim_other = 0;
    // ---- prologue: units blockIdx.x and blockIdx.x + G, both images filled by everybody
    if (threadIdx.x == 0) {
        for (int b = 0; b < NB; ++b) { mbar_init(&sh.full[b], 33); sh.pend_ok[b] = 0; }
        sh.ended = 0;
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __shared__ int s_pro[kPMaxBuf][2];       // prologue: halo_lo and records of the first NB units
    if ((int)threadIdx.x < NB) {
        const int b = threadIdx.x, u = (int)blockIdx.x + b * G;
        PSlot S;
        S.tile = -1; S.lo = S.hi = S.cb = S.ce = S.half = S.sums = S.pad = 0;
        int tile = -1, hlo = 0, nh = 0;
        if (u < A.U.n_units && !pslot_describe(S, A.U, u, A.tiles, A.cell_start, A.ls, A.s_cap, A.ctrl, tile, hlo, nh)) nh = 0;
        sh.slot[b] = S;
        sh.next[b] = S.cb;
        sh.done[b] = 0;
        s_pro[b][0] = hlo;
        s_pro[b][1] = nh;
    }
    if ((int)threadIdx.x < NB) smem_f4[(size_t)threadIdx.x * A.img_cap] = make_float4(TBSMA_SENTINEL, TBSMA_SENTINEL, TBSMA_SENTINEL, 0.f);
    __syncthreads();
#pragma unroll 1
    for (int b = 0; b < NB; ++b) {
        const int tile = sh.slot[b].tile, hlo = s_pro[b][0], nh = s_pro[b][1];
        if (tile < 0 || nh <= 0) continue;
        const unsigned short *__restrict__ img = A.ls.img + (size_t)tile * A.ls.img_stride;
        float4 *sm = smem_f4 + (size_t)b * A.img_cap;
        for (int k0 = threadIdx.x; k0 < nh; k0 += 4 * kPThreads) {
            float4 rec[4];
            unsigned short at[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int k = k0 + u * kPThreads;
                if (k < nh) { at[u] = img[k]; rec[u] = A.src[hlo + k]; }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (k0 + u * kPThreads < nh) sm[at[u]] = rec[u];
        }
    }
    __syncthreads();
    // ---- the warps work through the units, each at its own pace
    unsigned dead = 0u;          // bit b: buffer b has run out of units (for good)
    bool bad = false;
    int b = -1, round = 0;       // buffer of unit k = k % NB, round = k / NB
#pragma unroll 1
    for (;;) {
        if (++b == NB) { b = 0; ++round; }
        if (dead >> b & 1u) {
            if (dead == (1u << NB) - 1u) break;
            continue;
        }
        if (round >= 1) mbar_wait(&sh.full[b], (unsigned)((round - 1) & 1));
        // (the unit's description stays in shared memory: the chunk loops have no register to spare)
        const volatile PSlot &S = sh.slot[b];
        if (S.tile < 0) { dead |= 1u << b; continue; }
        const float4 *sm = smem_f4 + (size_t)b * A.img_cap;
        for (int ch = next_chunk(&sh.next[b]); ch < S.ce; ch = next_chunk(&sh.next[b])) {
            const int i = S.lo + (ch << 5) + lane;
            const uint2 *__restrict__ nl = A.nl + (size_t)S.half * A.ls.nl_stride;
            const int *__restrict__ nn = A.nn + (size_t)S.half * A.ls.n_stride;
            double *part = s_part + (size_t)b * NQ * A.U.max_chunks;
            if (PASS == 0) {
                if (i >= S.hi) continue;
                // own record, count and the first three rows in ONE round trip: the rows are read whatever the count is (they
                // exist: kg >= 3) and dropped afterwards if the list is shorter
                const uint2 *row = nl + tbsma_lrow(i, A.ls.kg);
                uint2 q0 = __ldcs(row), q1 = __ldcs(row + TBSMA_LROW), q2 = __ldcs(row + 2 * TBSMA_LROW);
                const float4 pi = A.src[i];
                const int ng = ((nn[i] & 0xffff) + 3) >> 2;
                if (ng < 3) { q2 = make_uint2(0u, 0u); if (ng < 2) q1 = q2; if (ng < 1) q0 = q2; }
                f32x2 rho2 = pk(0.f, 0.f);
                auto group = [&](const uint2 jj) {
                    const float4 p0 = lds_rec(sm, jj.x & 0xffffu), p1 = lds_rec(sm, jj.x >> 16);
                    const float4 p2 = lds_rec(sm, jj.y & 0xffffu), p3 = lds_rec(sm, jj.y >> 16);
                    rho2 = rho_term2(pi, p0, p1, A.pc, rho2);
                    rho2 = rho_term2(pi, p2, p3, A.pc, rho2);
                };
                // three rows in flight; a row register is reloaded right AFTER its use (loaded before, the new value needs a
                // second register while the old one is live, and the move back at the loop's end waits for the load)
                int g = 0;
                for (; g + 3 <= ng; g += 3) {
                    group(q0); q0 = ld_row(row, g + 3, ng, A.n_pad);
                    group(q1); q1 = ld_row(row, g + 4, ng, A.n_pad);
                    group(q2); q2 = ld_row(row, g + 5, ng, A.n_pad);
                }
                if (g < ng) {
                    group(q0);
                    if (g + 1 < ng) group(q1);
                }
                float rho0, rho1;
                unpk(rho2, rho0, rho1);
                const float rho = rho0 + rho1;
                const float s = rho > 0.f ? 1.0f / sqrtf(rho) : 0.f;     // once per atom, IEEE (D:A5 for rho = 0)
                A.xs[i] = make_float4(pi.x, pi.y, pi.z, s);
            } else {
                double se = 0.0, sk = 0.0, sw[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
                if (i < S.hi) {
                    const uint2 *row = nl + tbsma_lrow(i, A.ls.kg);
                    // FOUR rows in flight here (the density pass: three): the returning rows queue behind the shared-memory
                    // gathers on the load / store data path, and the force pass has the longer queue
                    uint2 q0 = __ldcs(row), q1 = __ldcs(row + TBSMA_LROW), q2 = __ldcs(row + 2 * TBSMA_LROW);
                    uint2 q3 = __ldcs(row + 3 * TBSMA_LROW);
                    const float4 pi = A.src[i];
                    const int nni = nn[i];
                    if (KICK) asm volatile("prefetch.global.L2 [%0];" ::"l"(A.kk.vel + i));   // read at the end of the chunk
                    const int ng = ((nni & 0xffff) + 3) >> 2;
                    if (ng < 4) { q3 = make_uint2(0u, 0u); if (ng < 3) q2 = q3; if (ng < 2) q1 = q3; if (ng < 1) q0 = q3; }
                    const f32x2 z2 = pk(0.f, 0.f);
                    AccT a = {z2, z2, z2, z2, z2, z2, z2, z2, z2, z2};
                    auto group = [&](const uint2 jj) {
                        const float4 p0 = lds_rec(sm, jj.x & 0xffffu), p1 = lds_rec(sm, jj.x >> 16);
                        const float4 p2 = lds_rec(sm, jj.y & 0xffffu), p3 = lds_rec(sm, jj.y >> 16);
                        force_term2<VIRIAL>(pi, p0, p1, A.pc, a);
                        force_term2<VIRIAL>(pi, p2, p3, A.pc, a);
                    };
                    int g = 0;
                    for (; g + 4 <= ng; g += 4) {
                        group(q0); q0 = ld_row(row, g + 4, ng, A.n_pad);
                        group(q1); q1 = ld_row(row, g + 5, ng, A.n_pad);
                        group(q2); q2 = ld_row(row, g + 6, ng, A.n_pad);
                        group(q3); q3 = ld_row(row, g + 7, ng, A.n_pad);
                    }
                    if (g < ng) {
                        group(q0);
                        if (g + 1 < ng) group(q1);
                        if (g + 2 < ng) group(q2);
                    }
                    const float fx = sum2(a.fx), fy = sum2(a.fy), fz = sum2(a.fz);
                    const float sqrt_rho = pi.w > 0.f ? 1.0f / pi.w : 0.f;
                    const float ei = __fmaf_rn(sum2(a.er), A.pc.e_rep_scale, -sqrt_rho);   // Eq.1-3: E_R^i + E_B^i
                    A.force[i] = make_float4(fx, fy, fz, ei);
                    bad = bad || !isfinite(fx + fy + fz + ei);
                    se = (double)ei;
                    if (KICK && (nni >> 16) == 0) {       // final B of the step, dynamic atoms only
                        float4 v = A.kk.vel[i];
                        v.x = __fmaf_rn(A.kk.kick, fx, v.x);
                        v.y = __fmaf_rn(A.kk.kick, fy, v.y);
                        v.z = __fmaf_rn(A.kk.kick, fz, v.z);
                        A.kk.vel[i] = v;
                        sk = (double)(A.kk.ke_scale * (v.x * v.x + v.y * v.y + v.z * v.z));
                    }
                    if (VIRIAL) {
                        sw[0] = 0.5 * (double)sum2(a.wxx); sw[1] = 0.5 * (double)sum2(a.wyy); sw[2] = 0.5 * (double)sum2(a.wzz);
                        sw[3] = 0.5 * (double)sum2(a.wxy); sw[4] = 0.5 * (double)sum2(a.wxz); sw[5] = 0.5 * (double)sum2(a.wyz);
                    }
                }
                __syncwarp();
                se = warp_sum_d(se);
                if (KICK) sk = warp_sum_d(sk);
                if (VIRIAL) {
#pragma unroll
                    for (int q = 0; q < 6; ++q) sw[q] = warp_sum_d(sw[q]);
                }
                if (lane == 0) {
                    const int c = ch - S.cb;
                    part[c] = se;
                    part[A.U.max_chunks + c] = sk;
                    if (VIRIAL) {
#pragma unroll
                        for (int q = 0; q < 6; ++q) part[(size_t)((2 + q) % NQ) * A.U.max_chunks + c] = sw[q];
                    }
                }
            }
        }
        // ---- out of unit k.  The last warp out adds up the unit and refills the buffer with unit k + 2.
        __syncwarp();
        int last = 0;
        if (lane == 0) {
            __threadfence_block();
            const int cnt = atomicAdd(&sh.done[b], 1);
            last = cnt == kPWarps - 1 ? 1 : 0;
            if (cnt == 0) {      // first out: claim and describe the unit that comes to this buffer next
                int u = -1;
                if (!sh.ended) {
                    u = atomicAdd(A.claim, 1) + NB * G;
                    if (u >= A.U.n_units) { u = -1; sh.ended = 1; }
                }
                PSlot N;
                N.tile = -1; N.lo = N.hi = N.cb = N.ce = N.half = N.sums = N.pad = 0;
                int tile = -1, hlo = 0, nh = 0;
                if (u >= 0 && !pslot_describe(N, A.U, u, A.tiles, A.cell_start, A.ls, A.s_cap, A.ctrl, tile, hlo, nh)) nh = 0;
                sh.pend[b] = N;
                sh.pend_tile[b] = tile; sh.pend_hlo[b] = hlo; sh.pend_nh[b] = tile < 0 ? 0 : nh;
                __threadfence_block();
                sh.pend_ok[b] = 1;
            }
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (!last) continue;
        __threadfence_block();
        if (PASS == 1) {      // the unit's sums: chunks in chunk order (lane l takes chunks l, l + 32, ...; then a fixed tree)
            double *my_sums = A.cta_sums + 8 * (size_t)S.sums;
            double *part = s_part + (size_t)b * NQ * A.U.max_chunks;
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                double v = 0.0;
                for (int c = lane; c < S.ce - S.cb; c += 32) v += part[(size_t)q * A.U.max_chunks + c];
                v = warp_sum_d(v);
                if (lane == 0) my_sums[q] = v;
            }
        }
        int tile = -1, hlo = 0, nh = 0;
        if (lane == 0) {
            while (!sh.pend_ok[b]) { }       // (the first warp out left long ago)
            __threadfence_block();
            const PSlot N = sh.pend[b];
            tile = sh.pend_tile[b]; hlo = sh.pend_hlo[b]; nh = sh.pend_nh[b];
            sh.pend_ok[b] = 0;
            sh.slot[b] = N;
            sh.next[b] = N.cb;
            sh.done[b] = 0;
        }
        tile = __shfl_sync(0xffffffffu, tile, 0);
        hlo = __shfl_sync(0xffffffffu, hlo, 0);
        nh = __shfl_sync(0xffffffffu, nh, 0);
        fill_image_async(smem_f4 + (size_t)b * A.img_cap, A.src, A.ls.img + (size_t)(tile < 0 ? 0 : tile) * A.ls.img_stride, hlo, nh, &sh.full[b]);
        if (lane == 0) mbar_arrive(&sh.full[b]);       // releases the slot description written above
    }
    if (PASS == 1 && bad) atomicOr(A.ctrl + 1, (int)TBSMA_FLAG_NONFINITE);
    // (density pass) launched as a programmatic dependent of the filter kernel: see k_density_tile
    if (PASS == 0) asm volatile("griddepcontrol.wait;" ::: "memory");
}

// per-replica sums of the CTA sums, in tile order (tbsma_compute; inside an MD step k_finish_step does it)
__global__ void __launch_bounds__(256)
k_reduce_replicas(TileSums ts, int R)
{
    tbsma_reduce_replicas(ts, R);
}

// ---- inspection (parity tests, bench statistics) ----------------------------------------------
__device__ __forceinline__ unsigned entry_of(const uint2 *__restrict__ nl, int kg, int i, int k)
{
    const uint2 w = nl[tbsma_lrow(i, kg) + (size_t)(k >> 2) * TBSMA_LROW];
    const unsigned h = (k & 2) ? w.y : w.x;
    return (k & 1) ? (h >> 16) : (h & 0xffffu);
}

__global__ void k_get_neighbors_tile(const int *__restrict__ tag, const uint2 *__restrict__ nl0,
                                     const int *__restrict__ nn0,
                                     const int *__restrict__ tileof, const int *__restrict__ inv,
                                     int inv_stride, const int *__restrict__ atom_rep, const int *__restrict__ cur,
                                     size_t nl_stride, int *__restrict__ counts, int *__restrict__ list, int n,
                                     int n_pad, int kmax)
{
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int h = cur[atom_rep[i]];
        const uint2 *nl = nl0 + (size_t)h * nl_stride;
        const int *nn = nn0 + (size_t)h * n_pad;
        const int t = tag[i];
        const int cnt = nn[i] & 0xffff;
        counts[t] = cnt;
        for (int k = 0; k < cnt; ++k)
            list[(size_t)t * kmax + k] =
                tag[inv[(size_t)tileof[i] * inv_stride + (entry_of(nl, kmax >> 2, i, k) >> 4)]];
    }
}

__global__ void k_count_pairs_tile(const float4 *__restrict__ pos, const uint2 *__restrict__ nl0,
                                   const int *__restrict__ nn0,
                                   const int *__restrict__ tileof, const int *__restrict__ inv,
                                   int inv_stride, const int *__restrict__ atom_rep, const int *__restrict__ cur,
                                   size_t nl_stride, unsigned long long *__restrict__ out, int n, int n_pad, float rc2, int kg,
                                   const RepGeom *__restrict__ geom)
{
    unsigned long long entries = 0, inside = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int h = cur[atom_rep[i]];
        const uint2 *nl = nl0 + (size_t)h * nl_stride;
        const int *nn = nn0 + (size_t)h * n_pad;
        const float4 pi = pos[i];
        const int cnt = nn[i] & 0xffff;
        entries += cnt;
        for (int k = 0; k < cnt; ++k) {
            const float4 pj = pos[inv[(size_t)tileof[i] * inv_stride + (entry_of(nl, kg, i, k) >> 4)]];
            float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
            {   // minimum image as D:A6 (a tile on a periodic boundary lists records from across it)
                const RepGeom *g = geom + atom_rep[i];
                if (g->periodic & 1) { const float hl = 0.5f * g->len[0]; if (dx > hl) dx -= g->len[0]; else if (dx < -hl) dx += g->len[0]; }
                if (g->periodic & 2) { const float hl = 0.5f * g->len[1]; if (dy > hl) dy -= g->len[1]; else if (dy < -hl) dy += g->len[1]; }
                if (g->periodic & 4) { const float hl = 0.5f * g->len[2]; if (dz > hl) dz -= g->len[2]; else if (dz < -hl) dz += g->len[2]; }
            }
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            inside += d2 < rc2;
        }
    }
    atomicAdd(out, entries);
    atomicAdd(out + 1, inside);
}

inline int grid_for(const tbsma_ctx *c, int64_t work, int threads, int per_sm)
{
    int64_t b = (work + threads - 1) / threads;
    const int64_t cap = (int64_t)c->n_sm * per_sm;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

size_t scan_smem(const tbsma_ctx *c)
{
    return (size_t)c->tile_cap * 16 + (size_t)c->tile_cell_cap * 4 + (size_t)c->tile_cap * 2;
}
int finish_threads(const tbsma_ctx *) { return kFinishMaxThreads; }
size_t finish_smem(const tbsma_ctx *c) { return (size_t)((c->tile_cap + 7) & ~7) * 2; }
size_t gather_smem(const tbsma_ctx *c) { return (size_t)c->img_cap * 16; }
size_t persist_smem(const tbsma_ctx *c, int pass, bool virial)
{
    return (size_t)c->p_nb * c->img_cap * 16 +
           (pass == 1 ? (size_t)c->p_nb * (virial ? 8 : 2) * c->p_max_chunks * sizeof(double) : 0);
}
size_t inner_smem(const tbsma_ctx *c) { return gather_smem(c) + (size_t)kInnerThreads * (c->kmax + 1) * 2; }
InnerArgs inner_args(const tbsma_ctx *c)
{
    InnerArgs ia;
    ia.olist = c->d_olist;
    ia.nn_o = c->d_nn_o;
    ia.nl = reinterpret_cast<uint2 *>(c->d_nlist);
    ia.nn = c->d_nn;
    ia.pos_build = c->d_pos_build;
    ia.cur = c->d_cur;
    ia.img = c->d_img;
    ia.img_stride = c->tile_cap;
    ia.img_cap = c->img_cap;
    ia.nl_stride = (size_t)(c->kmax / 4) * c->n_pad;
    ia.n_stride = c->n_pad;
    ia.pos_outer = c->d_pos_outer;
    ia.want_outer = c->d_want_outer;
    ia.kmax = c->kmax;
    ia.kg_o = c->kmax_o / 4;
    ia.rl2 = c->pc.rl2;
    // candidates are valid while no atom moved more than S/2 since their build (viol2).  New ones are asked
    // for one rebuild early: by the NEXT rebuild an atom moves at most skin/2 (+ one step) further.
    const double half_s = 0.5 * c->outer_skin, want = half_s - 0.5 * c->skin - 0.05;
    ia.viol2 = (float)(half_s * half_s);
    ia.want2 = want > 0.0 ? (float)(want * want) : -1.f;   // S too small to wait: every rebuild redoes the candidates
    return ia;
}

}  // namespace

// box shapes tried for a replica whose layers do not fit an image (or that is periodic), best own / halo ratio first
static const int kBoxCand[][3] = {{3, 3, 3}, {3, 3, 2}, {3, 2, 2}, {2, 2, 2}, {3, 3, 1}, {2, 2, 1}, {2, 1, 1}, {1, 1, 1}};
constexpr int kNBoxCand = sizeof(kBoxCand) / sizeof(kBoxCand[0]);

// own box b (clipped to the grid) of candidate cand for replica geometry g; false if a periodic axis is too short for it
// (a tile must not see a cell twice and must wrap at one end of an axis only: nc >= b + 2, see TileDesc)
static bool box_dims(const RepGeom &g, int cand, int b[3])
{
    for (int a = 0; a < 3; ++a) {
        b[a] = kBoxCand[cand][a] < g.nc[a] ? kBoxCand[cand][a] : g.nc[a];
        if ((g.periodic >> a & 1) && g.nc[a] < b[a] + 2) return false;
    }
    return true;
}

namespace {
// largest halo and own population over the box tiles of replica r for every candidate shape: out[(r * ncand + c) * 2 + {0, 1}]
__global__ void __launch_bounds__(128)
k_box_measure(const RepGeom *__restrict__ geom, const int *__restrict__ cell_start, int *__restrict__ out, int ncand)
{
    __shared__ int s_max[2];
    const int r = blockIdx.x, cnd = blockIdx.y;
    const RepGeom *g = geom + r;
    if (threadIdx.x < 2) s_max[threadIdx.x] = 0;
    __syncthreads();
    const int cand[8][3] = {{3, 3, 3}, {3, 3, 2}, {3, 2, 2}, {2, 2, 2}, {3, 3, 1}, {2, 2, 1}, {2, 1, 1}, {1, 1, 1}};
    int b[3], nt[3];
    bool ok = true;
    for (int a = 0; a < 3; ++a) {
        b[a] = min(cand[cnd][a], g->nc[a]);
        if ((g->periodic >> a & 1) && g->nc[a] < b[a] + 2) ok = false;
        nt[a] = (g->nc[a] + b[a] - 1) / b[a];
    }
    int mh = 0, mo = 0;
    if (ok) {
        const int ntile = nt[0] * nt[1] * nt[2];
        for (int ti = threadIdx.x; ti < ntile; ti += blockDim.x) {
            const int t3[3] = {ti % nt[0], (ti / nt[0]) % nt[1], ti / (nt[0] * nt[1])};
            int h0[3], hn[3], o0[3], on[3];
            for (int a = 0; a < 3; ++a) {
                o0[a] = t3[a] * b[a];
                on[a] = min(b[a], g->nc[a] - o0[a]);
                if (g->periodic >> a & 1) { h0[a] = o0[a] - 1; hn[a] = on[a] + 2; }
                else { h0[a] = max(o0[a] - 1, 0); hn[a] = min(o0[a] + on[a] + 1, g->nc[a]) - h0[a]; }
            }
            int nh = 0, no = 0;
            for (int z = 0; z < hn[2]; ++z)
                for (int y = 0; y < hn[1]; ++y)
                    for (int x = 0; x < hn[0]; ++x) {
                        const int cx = wrap_cell(h0[0] + x, g->nc[0]), cy = wrap_cell(h0[1] + y, g->nc[1]);
                        const int cz = wrap_cell(h0[2] + z, g->nc[2]);
                        const int cc = g->cell_base + (cz * g->nc[1] + cy) * g->nc[0] + cx;
                        const int pop = cell_start[cc + 1] - cell_start[cc];
                        nh += pop;
                        const int ax = h0[0] + x, ay = h0[1] + y, az = h0[2] + z;
                        if (ax >= o0[0] && ax < o0[0] + on[0] && ay >= o0[1] && ay < o0[1] + on[1] && az >= o0[2] &&
                            az < o0[2] + on[2])
                            no += pop;
                    }
            mh = max(mh, nh);
            mo = max(mo, no);
        }
    } else {
        mh = 0x7fffffff;
    }
    atomicMax(&s_max[0], mh);
    atomicMax(&s_max[1], mo);
    __syncthreads();
    if (threadIdx.x < 2) out[((size_t)r * ncand + cnd) * 2 + threadIdx.x] = s_max[threadIdx.x];
}
}  // namespace

// Sizes the tiles of every replica from the cells just binned.  A thin non-periodic replica (the paper's wires) is cut
// into runs of whole z-layers (kind 0): L_r own layers per tile, the largest L <= tile_layers whose halo (L + 2 layers of
// the replica's most populated layer, + 25 %) fits the shared-memory image.  Any other replica (thick wires, periodic
// bulk) is cut into boxes of cells (kind 1), the shape with the best own / halo ratio whose fullest halo, measured on the
// cells as they are, fits with 2.5 % to spare.  The choice depends on replica r alone, so a replica is tiled (and therefore
// summed) identically whatever batch it is part of.  Returns TBSMA_OK and sets active_variant = 2, or leaves
// active_variant = 1 when a replica does not fit either way.
int tbsma_tile_setup(tbsma_ctx *c, cudaStream_t st)
{
    c->active_variant = 1;
    if (c->variant == 1 || c->n == 0) return TBSMA_OK;
    if (c->kmax_o > 248 || !c->d_olist) return c->variant == 2 ? TBSMA_EINVAL : TBSMA_OK;
    const int R = c->R;
    k_layer_maxpop<<<(R + 127) / 128, 128, 0, st>>>(c->d_geom, c->d_cell_start, c->d_maxpop, R);
    c->launches++;
    int *maxpop = (int *)malloc(sizeof(int) * 2 * R);
    if (!maxpop) return TBSMA_ENOMEM;
    cudaError_t e = cudaMemcpyAsync(maxpop, c->d_maxpop, sizeof(int) * 2 * R, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) { free(maxpop); return TBSMA_ECUDA; }
    const int cap = TBSMA_TILE_MAX_RECORDS;
    int lmax = c->tile_layers;
    if (lmax < 1) lmax = 1;
    if (lmax > TBSMA_TILE_MAX_LAYERS) lmax = TBSMA_TILE_MAX_LAYERS;
    int64_t n_tiles = 0;
    int cell_cap = 0, rec_cap = 0, own_cap = 0, box_min = 0, box_want = 0;
    bool fits = true, any_box = false;
    int *Lr = (int *)malloc(sizeof(int) * R);      // > 0: own layers per tile (kind 0); <= 0: -(box candidate) (kind 1)
    if (!Lr) { free(maxpop); return TBSMA_ENOMEM; }
    for (int r = 0; r < R; ++r) {
        const RepGeom &g = c->h_geom[r];
        const int64_t pop = ((int64_t)maxpop[r] * 5 + 3) / 4 + 1;    // + 25 % for later rebuilds
        int L = (int)(cap / pop) - 2;
        if (L > lmax) L = lmax;
        const int lc = g.nc[0] * g.nc[1];
        if (g.periodic || c->tile_force_box || L < 1 || (int64_t)(L + 2) * lc + 1 > 8192) { Lr[r] = 0; any_box = true; continue; }
        if ((L + 2) * lc + 1 > cell_cap) cell_cap = (L + 2) * lc + 1;
        if ((int)((L + 2) * pop) > rec_cap) rec_cap = (int)((L + 2) * pop);
        if ((int)(L * pop) > own_cap) own_cap = (int)(L * pop);
        Lr[r] = L;
        n_tiles += (g.nc[2] + L - 1) / L;
    }
    free(maxpop);
    if (any_box) {
        // measure every candidate shape on the cells as they are, take the best that fits
        int *d_meas = nullptr;
        const size_t nm = (size_t)R * kNBoxCand * 2;
        int *meas = (int *)malloc(sizeof(int) * nm);
        if (!meas) { free(Lr); return TBSMA_ENOMEM; }
        e = cudaMalloc((void **)&d_meas, sizeof(int) * nm);
        if (e == cudaSuccess) {
            k_box_measure<<<dim3(R, kNBoxCand), 128, 0, st>>>(c->d_geom, c->d_cell_start, d_meas, kNBoxCand);
            c->launches++;
            e = cudaMemcpyAsync(meas, d_meas, sizeof(int) * nm, cudaMemcpyDeviceToHost, st);
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        cudaFree(d_meas);
        if (e != cudaSuccess) { free(meas); free(Lr); return TBSMA_ECUDA; }
        for (int r = 0; r < R && fits; ++r) {
            if (Lr[r] > 0) continue;
            const RepGeom &g = c->h_geom[r];
            int pick = -1;
            for (int cnd = 0; cnd < kNBoxCand && pick < 0; ++cnd) {
                int b[3];
                if (!box_dims(g, cnd, b)) continue;
                int hc = 1;
                for (int a = 0; a < 3; ++a) hc *= (g.periodic >> a & 1) ? b[a] + 2 : (b[a] + 2 < g.nc[a] ? b[a] + 2 : g.nc[a]);
                if (hc > TBSMA_TILE_MAX_RUNS || b[0] * b[1] * b[2] > TBSMA_TILE_MAX_OWN_RUNS) continue;
                const int64_t mh = meas[((size_t)r * kNBoxCand + cnd) * 2];
                if (mh + mh / 40 + 8 > cap) continue;
                pick = cnd;
            }
            if (pick < 0) { fits = false; break; }
            Lr[r] = -pick;
            int b[3];
            box_dims(g, pick, b);
            const int mh = meas[((size_t)r * kNBoxCand + pick) * 2], mo = meas[((size_t)r * kNBoxCand + pick) * 2 + 1];
            // A candidate is taken when its halo fits with 2.5 % to spare; the image is then sized with up to 10 %
            // (below): later rebuilds of the cells inside tbsma_md_run (a thick wire strained or compressed, atoms
            // diffusing between cells) cannot resize it.
            if (mh + mh / 40 + 8 > box_min) box_min = mh + mh / 40 + 8;
            int want = mh + mh / 10 + 8;
            if (want > cap) want = cap;
            if (want > box_want) box_want = want;
            if (mo + mo / 20 + 16 > own_cap) own_cap = mo + mo / 20 + 16;
            n_tiles += (int64_t)((g.nc[0] + b[0] - 1) / b[0]) * ((g.nc[1] + b[1] - 1) / b[1]) * ((g.nc[2] + b[2] - 1) / b[2]);
        }
        free(meas);
        if (fits && box_min > 0) {
            // Image size of the box tiles: between what the 2.5 % rule needs and 10 % headroom, the largest that costs
            // no CTA per SM in the kernels whose residency the image decides (the list filter, whose shared memory is the
            // image plus a column per thread, and the gather passes).  Measured on the 64^3 block: 10 % regardless took
            // the filter kernel from two CTAs per SM to one and the list renewal from 0.153 to 0.219 ms per step.
            int per_sm = 0, dev = 0;
            cudaFuncAttributes fa_inner = {}, fa_gather = {};
            e = cudaGetDevice(&dev);
            if (e == cudaSuccess) e = cudaDeviceGetAttribute(&per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev);
            if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa_inner, k_tile_inner);
            if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa_gather, k_force_tile<false, true, false>);
            if (e != cudaSuccess) { free(Lr); return TBSMA_ECUDA; }
            auto img_of = [](int rec) {
                int img = rec + rec / 8 + 64 + 1;
                if (img > TBSMA_TILE_MAX_RECORDS + 1) img = TBSMA_TILE_MAX_RECORDS + 1;
                return img < rec + 1 ? rec + 1 : img;
            };
            auto resident = [&](int rec, int which) {
                const size_t dyn = (size_t)img_of(rec) * 16 + (which == 0 ? (size_t)kInnerThreads * (c->kmax + 1) * 2 : 0);
                const size_t stat = which == 0 ? fa_inner.sharedSizeBytes : fa_gather.sharedSizeBytes;
                return (int)((size_t)per_sm / (dyn + stat + 1024));
            };
            const int lo = rec_cap > box_min ? rec_cap : box_min, hi = box_want > lo ? box_want : lo;
            int pick = lo;
            for (int rcand = hi; rcand > lo; rcand -= 8)
                if (resident(rcand, 0) == resident(lo, 0) && resident(rcand, 1) == resident(lo, 1)) { pick = rcand; break; }
            rec_cap = pick;
        }
    }
    if (!fits || n_tiles > 0x7fffffff) {
        free(Lr);
        return c->variant == 2 ? TBSMA_EINVAL : TBSMA_OK;   // forced tile variant that does not fit
    }
    // A box tile stages eight halo records per own atom (a wire's layer tile: two and a half) and holds few chunks of
    // work; measured, box tiles beat the global gather on the 10^6-atom periodic block (2 197 tiles: 1.92 against 1.74 G
    // atom-steps/s) and lose to it on the 165 000-atom thick wire (882 tiles: 1.18 against 1.77 G).  Left to itself
    // (variant 0) the library takes them for large batches only.
    if (c->variant == 0 && any_box && n_tiles < 8 * (int64_t)c->n_sm) { free(Lr); return TBSMA_OK; }
    c->any_box = any_box ? 1 : 0;
    TileDesc *h = (TileDesc *)calloc((size_t)(n_tiles ? n_tiles : 1), sizeof(TileDesc));
    int *first = (int *)malloc(sizeof(int) * (size_t)(R + 1));
    if (!h || !first) { free(Lr); free(h); free(first); return TBSMA_ENOMEM; }
    int64_t k = 0;
    for (int r = 0; r < R; ++r) {
        first[r] = (int)k;
        const RepGeom &g = c->h_geom[r];
        const int lc = g.nc[0] * g.nc[1], nz = g.nc[2], L = Lr[r];
        if (L > 0) {
            for (int z0 = 0; z0 < nz; z0 += L) {
                const int z1 = z0 + L < nz ? z0 + L : nz;
                const int zh0 = z0 > 0 ? z0 - 1 : 0, zh1 = z1 < nz ? z1 + 1 : nz;
                TileDesc &t = h[k++];
                t.rep = r;
                t.kind = 0;
                t.first_of_rep = z0 == 0;
                t.ch0 = g.cell_base + zh0 * lc;
                t.nlay_h = zh1 - zh0;
                t.own_first = z0 - zh0;
                t.own_n = z1 - z0;
                t.layer_cells = lc;
                t.nx = g.nc[0]; t.ny = g.nc[1]; t.nz = nz;
                t.z_h0 = zh0;
                t.cell_base = g.cell_base;
                for (int a = 0; a < 3; ++a) { t.Ls[a] = 0.f; t.hL[a] = INFINITY; }
            }
            continue;
        }
        int b[3];
        box_dims(g, -L, b);
        const int64_t k0 = k;
        for (int oz = 0; oz < g.nc[2]; oz += b[2])
            for (int oy = 0; oy < g.nc[1]; oy += b[1])
                for (int ox = 0; ox < g.nc[0]; ox += b[0]) {
                    TileDesc &t = h[k++];
                    t.rep = r;
                    t.kind = 1;
                    t.first_of_rep = k - 1 == k0;
                    t.cell_base = g.cell_base;
                    t.nx = g.nc[0]; t.ny = g.nc[1]; t.nz = g.nc[2];
                    const int o[3] = {ox, oy, oz};
                    for (int a = 0; a < 3; ++a) {
                        const int on = b[a] < g.nc[a] - o[a] ? b[a] : g.nc[a] - o[a];
                        int h0, hn;
                        t.Ls[a] = 0.f;
                        t.hL[a] = INFINITY;
                        if (g.periodic >> a & 1) {
                            h0 = o[a] - 1;
                            hn = on + 2;
                            if (h0 < 0) { t.Ls[a] = g.len[a]; t.hL[a] = 0.5f * g.len[a]; }                    // lower end
                            else if (h0 + hn > g.nc[a]) { t.Ls[a] = -g.len[a]; t.hL[a] = 0.5f * g.len[a]; }   // upper end
                        } else {
                            h0 = o[a] > 0 ? o[a] - 1 : 0;
                            hn = (o[a] + on + 1 < g.nc[a] ? o[a] + on + 1 : g.nc[a]) - h0;
                        }
                        t.h0[a] = (short)h0; t.hn[a] = (short)hn; t.o0[a] = (short)(o[a] - h0); t.on[a] = (short)on;
                    }
                }
    }
    first[R] = (int)k;
    free(Lr);
    // the tables keep their allocations from one tbsma_build_cells to the next while they are large enough
    // (tbsma_md_run_host rebuilds the cells in every call)
    auto ensure = [](void **p, size_t *have, size_t need) -> cudaError_t {
        if (*p && *have >= need) return cudaSuccess;
        cudaFree(*p);
        *p = nullptr;
        *have = 0;
        const cudaError_t err = cudaMalloc(p, need);
        if (err == cudaSuccess) *have = need;
        return err;
    };
    const size_t nt1 = (size_t)(n_tiles ? n_tiles : 1);
    const int new_tile_cap = rec_cap < cap ? rec_cap : cap;
    int new_img_cap = new_tile_cap + new_tile_cap / 8 + 64 + 1;
    if (new_img_cap > TBSMA_TILE_MAX_RECORDS + 1) new_img_cap = TBSMA_TILE_MAX_RECORDS + 1;
    if (new_img_cap < new_tile_cap + 1) new_img_cap = new_tile_cap + 1;
    e = ensure((void **)&c->d_tiles, &c->have_tiles, sizeof(TileDesc) * nt1);
    if (e == cudaSuccess) e = ensure((void **)&c->d_tile_first, &c->have_first, sizeof(int) * (size_t)(R + 1));
    if (e == cudaSuccess) e = ensure((void **)&c->d_work, &c->have_work, sizeof(int) * (size_t)(2 + 2 * n_tiles));
    if (e == cudaSuccess) e = ensure((void **)&c->d_img, &c->have_img, sizeof(unsigned short) * nt1 * new_tile_cap);
    if (e == cudaSuccess) e = ensure((void **)&c->d_inv, &c->have_inv, sizeof(int) * nt1 * new_img_cap);
    // Few tiles (one or a few small wires): several CTAs share a tile, each filling the image and taking a share of the
    // 32-atom chunks, until the CTAs fill the GPU about twice (or every CTA is down to one chunk).
    int nsplit = 1;
    {
        const int slots = 8 * c->n_sm;
        int est_chunks = (own_cap * 4 / 5 + 31) / 32;     // own_cap carries 25 % headroom
        if (est_chunks < 1) est_chunks = 1;
        // (box tiles hold few chunks and cost a large image each: they are split only when there are very few of them)
        if (n_tiles > 0 && n_tiles < (any_box ? slots / 4 : slots)) nsplit = (int)((slots + n_tiles - 1) / n_tiles);
        if (nsplit > est_chunks) nsplit = est_chunks;
        if (c->tile_split_req > 0) nsplit = c->tile_split_req;
        if (nsplit < 1) nsplit = 1;
    }
    // Units of the persistent gather kernels (k_gather_persist): whole tiles, except that the LAST tiles of the pass are
    // cut into S parts so that the CTAs run out of work together, and that batches with few tiles are cut throughout.
    int pS = 1, p_plain = (int)n_tiles;
    {
        const int G = 2 * c->n_sm;
        int est_chunks = (own_cap * 4 / 5 + 31) / 32;
        if (est_chunks < 1) est_chunks = 1;
        if (c->tile_split_req > 0) { pS = c->tile_split_req; p_plain = 0; }
        else if (n_tiles < 4 * (int64_t)G) {
            pS = n_tiles > 0 ? (int)((4 * (int64_t)G + n_tiles - 1) / n_tiles) : 1;
            if (pS > est_chunks) pS = est_chunks;
            p_plain = 0;
        } else {
            // many tiles per CTA: whole tiles (a split tile is filled once per part, and the parts are too short to hide it)
            pS = c->p_tail_split > 0 ? c->p_tail_split : 1;
            if (pS > est_chunks) pS = est_chunks;
            p_plain = (int)n_tiles - G;
        }
        if (pS < 1) pS = 1;
        if (pS == 1) p_plain = (int)n_tiles;
    }
    c->p_S = pS;
    c->p_plain = p_plain;
    c->p_units = p_plain + ((int)n_tiles - p_plain) * pS;
    c->p_max_chunks = (own_cap + 31) / 32 + 2;
    const size_t sums_slots = nt1 * (size_t)(nsplit > pS ? nsplit : pS);
    if (e == cudaSuccess) e = ensure((void **)&c->d_cta_sums, &c->have_sums, sizeof(double) * 8 * sums_slots);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->d_cta_sums, 0, sizeof(double) * 8 * sums_slots, st);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->d_work, 0, sizeof(int) * (size_t)(2 + 2 * n_tiles), st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_tiles, h, sizeof(TileDesc) * (size_t)n_tiles, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaMemcpyAsync(c->d_tile_first, first, sizeof(int) * (size_t)(R + 1), cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    free(h);
    free(first);
    if (e != cudaSuccess) return e == cudaErrorMemoryAllocation ? TBSMA_ENOMEM : TBSMA_ECUDA;
    c->n_tiles = (int)n_tiles;
    c->tile_nsplit = nsplit;
    c->tile_cap = new_tile_cap;   // halo records a tile may hold
    // image: the sentinel + eight colour classes of records (k_tile_place); room for classes 1/8 + 64 fuller than even
    c->img_cap = new_img_cap;
    c->tile_cell_cap = (cell_cap + 3) & ~3;
    c->own_cap = own_cap;
    // opt in to > 48 KB of dynamic shared memory
    const int sm_scan = (int)scan_smem(c), sm_fin = (int)finish_smem(c), sm_g = (int)gather_smem(c);
    e = cudaFuncSetAttribute(k_tile_scan, cudaFuncAttributeMaxDynamicSharedMemorySize, sm_scan);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(k_tile_inner, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)inner_smem(c));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_tile_finish, cudaFuncAttributeMaxDynamicSharedMemorySize, sm_fin);
#define TBSMA_ATTR(K) if (e == cudaSuccess) e = cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, sm_g)
    TBSMA_ATTR(k_density_tile<false>); TBSMA_ATTR(k_density_tile<true>);
    TBSMA_ATTR((k_force_tile<false, false, false>)); TBSMA_ATTR((k_force_tile<false, true, false>));
    TBSMA_ATTR((k_force_tile<true, false, false>)); TBSMA_ATTR((k_force_tile<true, true, false>));
    TBSMA_ATTR((k_force_tile<false, false, true>)); TBSMA_ATTR((k_force_tile<false, true, true>));
    TBSMA_ATTR((k_force_tile<true, false, true>)); TBSMA_ATTR((k_force_tile<true, true, true>));
#undef TBSMA_ATTR
    {
        // image buffers per CTA: as many (up to the requested depth) as let two CTAs share an SM
        c->p_nb = c->p_nb_req > 0 ? c->p_nb_req : 2;     // (3 measured no faster than 2 on config 3)
        if (c->p_nb > kPMaxBuf) c->p_nb = kPMaxBuf;
        while (c->p_nb > 2 && persist_smem(c, 1, true) > 112 * 1024) c->p_nb--;
        const int sm_p0 = (int)persist_smem(c, 0, false), sm_p1 = (int)persist_smem(c, 1, false), sm_p1v = (int)persist_smem(c, 1, true);
#define TBSMA_ATTR(K, B) if (e == cudaSuccess) e = cudaFuncSetAttribute(K, cudaFuncAttributeMaxDynamicSharedMemorySize, B)
        TBSMA_ATTR((k_gather_persist<0, false, false>), sm_p0);
        TBSMA_ATTR((k_gather_persist<1, false, false>), sm_p1); TBSMA_ATTR((k_gather_persist<1, false, true>), sm_p1);
        TBSMA_ATTR((k_gather_persist<1, true, false>), sm_p1v); TBSMA_ATTR((k_gather_persist<1, true, true>), sm_p1v);
#undef TBSMA_ATTR
        c->persist_ok = sm_p1v <= 112 * 1024 && c->kmax >= 16;     // two CTAs per SM; four rows per atom exist
    }
    {   // the fused step of small batches: every CTA of the grid must be resident at once (cooperative launch)
        int occ = 0, min_occ = 1 << 30;
#define TBSMA_FUSED(V, S)                                                                                                     \
        if (e == cudaSuccess) e = cudaFuncSetAttribute(k_step_small<V, S>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm_g);   \
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_step_small<V, S>, 256, (size_t)sm_g);     \
        if (occ < min_occ) min_occ = occ;
        TBSMA_FUSED(false, false) TBSMA_FUSED(false, true) TBSMA_FUSED(true, false) TBSMA_FUSED(true, true)
#undef TBSMA_FUSED
        c->fused_max_ctas = e == cudaSuccess ? min_occ * c->n_sm : 0;
        // a batch that would fit the fused step with fewer parts per tile gets fewer parts -- whether or not the fused step
        // is switched on: the parts fix the grouping of the per-replica fp64 sums, and tbsma_set_fused_step promises to
        // change cost only, whenever it is called
        if (c->tile_split_req <= 0 && c->n_tiles <= c->fused_max_ctas &&
            (int64_t)c->n_tiles * c->tile_nsplit > c->fused_max_ctas)
            c->tile_nsplit = c->fused_max_ctas / c->n_tiles;
    }
    if (e != cudaSuccess) return TBSMA_ECUDA;
    c->active_variant = 2;
    return TBSMA_OK;
}

// K1 -> K2 -> K3 for the dirty replicas; expects cell-ordered pos / vel / tag in the tmp buffers
cudaError_t tbsma_launch_tile_lists(tbsma_ctx *c, float4 *pos, float4 *vel, int32_t *tag, cudaStream_t st)
{
    const int n = (int)c->n;
    const DirtyView dv = tbsma_dirty_view(c);
    uint2 *ol = c->d_olist;
    uint2 *ol_tmp = ol + (size_t)(c->kmax_o / 4) * c->n_pad;    // second half of the allocation
    ScanArgs sa;
    sa.cell_start = c->d_cell_start; sa.cell_sorted = c->d_slot; sa.ctrl = c->d_ctrl; sa.pos_sorted = c->d_tmp_pos;
    sa.nl_tmp = ol_tmp; sa.nn_tmp = c->d_nn_tmp; sa.newslot = c->d_newslot; sa.oldof = c->d_oldof;
    sa.want_outer = c->d_want_outer; sa.n_pad = c->n_pad; sa.kmax = c->kmax_o; sa.ro2 = c->pc.ro2; sa.rl2 = c->pc.rl2;
    sa.s_cap = c->tile_cap; sa.cell_cap = c->tile_cell_cap;
    FinishArgs fa;
    fa.cell_start = c->d_cell_start; fa.nl_tmp = ol_tmp; fa.nn_tmp = c->d_nn_tmp; fa.newslot = c->d_newslot;
    fa.oldof = c->d_oldof; fa.nl = ol; fa.nn = c->d_nn_o; fa.tileof = c->d_tileof;
    fa.img = c->d_img; fa.img_stride = c->tile_cap; fa.n_pad = c->n_pad; fa.kg_o = c->kmax_o / 4;
    fa.s_cap = c->tile_cap;
    PlaceArgs pa;
    pa.cell_start = c->d_cell_start; pa.oldof = c->d_oldof; pa.pos_sorted = c->d_tmp_pos; pa.geom = c->d_geom;
    pa.img = c->d_img; pa.inv = c->d_inv; pa.img_stride = c->tile_cap; pa.inv_stride = c->img_cap;
    pa.img_cap = c->img_cap; pa.inv_h = c->balance && c->class_h > 0.0 ? (float)(1.0 / c->class_h) : 0.f;
    pa.ctrl = c->d_ctrl;
    const int gw = c->n_tiles < 2 * c->n_sm ? c->n_tiles : 2 * c->n_sm;
    k_tile_scan<<<gw, kScanThreads, scan_smem(c), st>>>(c->d_tiles, c->d_work, c->n_tiles, sa);
    k_tile_place<<<gw, 256, 0, st>>>(c->d_tiles, c->d_work, c->n_tiles, pa);
    k_tile_finish<<<gw, finish_threads(c), finish_smem(c), st>>>(c->d_tiles, c->d_work, c->n_tiles, fa);
    k_tile_permute<<<grid_for(c, n, 256, 8), 256, 0, st>>>(pos, vel, tag, c->d_pos_outer, c->d_atom_rep, dv,
                                                          c->d_oldof, c->d_tmp_pos, c->d_tmp4, c->d_tmp_tag, n);
    c->launches += 4;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_tile_worklist(tbsma_ctx *c, cudaStream_t st, unsigned long long cond, int use_cond)
{
    k_tile_worklist<<<1, 256, 0, st>>>(c->d_dirty, c->d_tile_first, c->d_work, c->R, c->n_tiles,
                                       (cudaGraphConditionalHandle)cond, use_cond, c->d_ctrl + 4);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_tile_inner(tbsma_ctx *c, const float4 *pos, int which, cudaStream_t st, bool beside)
{
    int nsplit = (c->own_cap + kInnerThreads - 1) / kInnerThreads;
    if (nsplit < 1) nsplit = 1;
    const int64_t units = (int64_t)c->n_tiles * nsplit;
    const size_t sm = inner_smem(c);
    // Beside the gather passes of the step (their kernels fill the register file: a filter CTA on an SM keeps a gather CTA
    // off it) the pass gets ONE CTA per SM; measured against two: config 4 1.0081 -> 0.9941 ms, config 3 0.5208 -> 0.5186 ms
    // per step.  Run on its own (first build, fixed cadence, new candidates) it takes what fits.
    int per_sm = 1;
    if (!beside && cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_tile_inner, kInnerThreads, sm) != cudaSuccess) per_sm = 1;
    if (per_sm > 4) per_sm = 4;
    if (per_sm < 1) per_sm = 1;
    const int64_t cap = (int64_t)per_sm * c->n_sm;
    const int grid = (int)(units < cap ? units : cap);
    k_tile_inner<<<grid, kInnerThreads, sm, st>>>(c->d_tiles, c->d_work, c->d_cell_start, pos, inner_args(c), c->d_ctrl,
                                                  c->n_pad, c->tile_cap, nsplit, which, c->n_tiles);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_stage_copy(tbsma_ctx *c, const float4 *pos, const float4 *vel, const int32_t *tag,
                                    cudaStream_t st)
{
    k_stage_copy<<<grid_for(c, c->n, 256, 8), 256, 0, st>>>(pos, vel, tag, c->d_tmp_pos, c->d_tmp4, c->d_tmp_tag, (int)c->n);
    c->launches++;
    return cudaGetLastError();
}

static ListSel list_sel(const tbsma_ctx *c, int sync_level)
{
    ListSel ls;
    ls.cur = c->d_cur;
    ls.dirty = c->d_dirty;
    ls.sync_level = sync_level;
    ls.nl_stride = (size_t)(c->kmax / 4) * c->n_pad;
    ls.n_stride = c->n_pad;
    ls.img = c->d_img;
    ls.img_stride = c->tile_cap;
    ls.nsplit = c->tile_nsplit;
    ls.kg = c->kmax / 4;
    return ls;
}

// persistent kernels for batches with at least two tiles per CTA (or when asked for by depth, tbsma_set_gather(2..4));
// a handful of tiles (one small wire) is quicker with one short-lived CTA per part of a tile
static bool use_persist(const tbsma_ctx *c)
{
    return c->gather_mode != 0 && c->persist_ok && !c->any_box && (c->p_nb_req > 0 || c->n_tiles >= 4 * c->n_sm);
}

static PArgs persist_args(tbsma_ctx *c, int pass, const float4 *src, int sync_level)
{
    PArgs A;
    A.tiles = c->d_tiles; A.cell_start = c->d_cell_start; A.src = src;
    A.nl = reinterpret_cast<const uint2 *>(c->d_nlist); A.nn = c->d_nn;
    A.xs = c->d_xs; A.force = nullptr; A.cta_sums = c->d_cta_sums;
    A.kk.vel = nullptr; A.kk.kick = 0.f; A.kk.ke_scale = 0.f; A.kk.ekin = nullptr;
    A.ctrl = c->d_ctrl; A.claim = c->d_ctrl + 4 + pass; A.claim_other = c->d_ctrl + 4 + (pass ^ 1);
    A.ls = list_sel(c, sync_level);
    A.n_pad = c->n_pad; A.s_cap = c->tile_cap; A.img_cap = c->img_cap;
    A.nb = c->p_nb;
    A.U.n_units = c->p_units; A.U.n_plain = c->p_plain; A.U.S = c->p_S; A.U.max_chunks = c->p_max_chunks;
    A.pc = c->pc;
    return A;
}
static int persist_grid(const tbsma_ctx *c)
{
    const int G = 2 * c->n_sm;
    return c->p_units < G ? (c->p_units > 0 ? c->p_units : 1) : G;
}

// early: the launch may begin while the kernel before it on the stream (the filter pass of the replicas renewing
// their lists, whose output this launch does not read) is still running: programmatic dependent launch
cudaError_t tbsma_launch_density_tile(tbsma_ctx *c, const float4 *pos, int sync_level, cudaStream_t st, bool early)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(c->n_tiles * c->tile_nsplit));
    cfg.blockDim = dim3(c->tile_threads);
    cfg.dynamicSmemBytes = gather_smem(c);
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = early ? 1 : 0;
    if (use_persist(c)) {
        // Both passes' unit counters start at zero without relying on the previous pair of passes having run to its end.
        // An early launch is a programmatic dependent of the filter kernel (nothing may sit between the two); it is only
        // used inside a step, whose k_tile_worklist has cleared the counters already.
        if (!early) {
            const cudaError_t em = cudaMemsetAsync(c->d_ctrl + 4, 0, 2 * sizeof(int), st);
            if (em != cudaSuccess) return em;
        }
        cfg.gridDim = dim3((unsigned)persist_grid(c));
        cfg.blockDim = dim3(kPThreads);
        cfg.dynamicSmemBytes = persist_smem(c, 0, false);
        const PArgs A = persist_args(c, 0, pos, sync_level);
        const cudaError_t ep = cudaLaunchKernelEx(&cfg, k_gather_persist<0, false, false>, A);
        c->launches++;
        return ep != cudaSuccess ? ep : cudaGetLastError();
    }
    const cudaError_t e =
        c->tile_nsplit > 1
            ? cudaLaunchKernelEx(&cfg, k_density_tile<true>, (const TileDesc *)c->d_tiles, (const int *)c->d_cell_start, pos,
                                 reinterpret_cast<const uint2 *>(c->d_nlist), (const int *)c->d_nn, c->d_xs, c->d_ctrl,
                                 list_sel(c, sync_level), c->n_pad, c->tile_cap, c->pc)
            : cudaLaunchKernelEx(&cfg, k_density_tile<false>, (const TileDesc *)c->d_tiles, (const int *)c->d_cell_start, pos,
                                 reinterpret_cast<const uint2 *>(c->d_nlist), (const int *)c->d_nn, c->d_xs, c->d_ctrl,
                                 list_sel(c, sync_level), c->n_pad, c->tile_cap, c->pc);
    c->launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t tbsma_launch_force_tile(tbsma_ctx *c, float4 *force, bool virial, KickArgs kk, int sync_level,
                                    cudaStream_t st)
{
    if (use_persist(c)) {
        PArgs A = persist_args(c, 1, c->d_xs, sync_level);
        A.force = force;
        A.kk = kk;
        const int g = persist_grid(c);
        const size_t sm = persist_smem(c, 1, virial);
        if (virial) {
            if (kk.vel) k_gather_persist<1, true, true><<<g, kPThreads, sm, st>>>(A);
            else k_gather_persist<1, true, false><<<g, kPThreads, sm, st>>>(A);
        } else {
            if (kk.vel) k_gather_persist<1, false, true><<<g, kPThreads, sm, st>>>(A);
            else k_gather_persist<1, false, false><<<g, kPThreads, sm, st>>>(A);
        }
        c->launches++;
        return cudaGetLastError();
    }
    const uint2 *nl = reinterpret_cast<const uint2 *>(c->d_nlist);
    const size_t sm = gather_smem(c);
    const int g = c->n_tiles * c->tile_nsplit, b = c->tile_threads;
    const ListSel ls = list_sel(c, sync_level);
#define TBSMA_FT(V, K, S)                                                                                          \
    k_force_tile<V, K, S><<<g, b, sm, st>>>(c->d_tiles, c->d_cell_start, c->d_xs, nl, c->d_nn, force, c->d_cta_sums, kk, \
                                            c->d_ctrl, ls, c->n_pad, c->tile_cap, c->pc)
#define TBSMA_FT2(V, K) do { if (c->tile_nsplit > 1) TBSMA_FT(V, K, true); else TBSMA_FT(V, K, false); } while (0)
    if (virial) { if (kk.vel) TBSMA_FT2(true, true); else TBSMA_FT2(true, false); }
    else        { if (kk.vel) TBSMA_FT2(false, true); else TBSMA_FT2(false, false); }
#undef TBSMA_FT2
#undef TBSMA_FT
    c->launches++;
    return cudaGetLastError();
}

// the whole step in one cooperative launch (k_step_small): small batches of the tile variant
bool tbsma_step_small_ok(const tbsma_ctx *c)
{
    return c->active_variant == 2 && c->fused_step && !use_persist(c) && c->tile_threads == 256 &&
           (int64_t)c->n_tiles * c->tile_nsplit <= c->fused_max_ctas && c->n_tiles > 0;
}

cudaError_t tbsma_launch_step_small(tbsma_ctx *c, float4 *pos, float4 *vel, float4 *force, const int32_t *tag,
                                    const StepArgs &a, KickArgs kk, bool virial, int advance_offset, TileSums ts,
                                    unsigned long long cond, cudaStream_t st)
{
    FusedArgs F;
    F.pos = pos; F.vel = vel; F.force = force; F.pos_build = c->d_pos_build; F.atom_rep = c->d_atom_rep; F.geom = c->d_geom;
    F.tag = tag; F.a = a; F.counters = c->d_counters; F.dirty = c->d_dirty; F.ctrl = c->d_ctrl; F.n = (int)c->n; F.R = c->R;
    F.tiles = c->d_tiles; F.cell_start = c->d_cell_start; F.nl = reinterpret_cast<const uint2 *>(c->d_nlist); F.nn = c->d_nn;
    F.xs = c->d_xs; F.cta_sums = c->d_cta_sums; F.kk = kk; F.ls = list_sel(c, 2); F.n_pad = c->n_pad; F.s_cap = c->tile_cap;
    F.pc = c->pc; F.stagger = c->d_stagger; F.cur = c->d_cur; F.swap = c->list_bufs == 2;
    F.advance = advance_offset & 1; F.count_step = (advance_offset >> 1) & 1; F.ts = ts;
    F.cond = (cudaGraphConditionalHandle)cond;
    void *args[] = {&F};
    const dim3 grid((unsigned)(c->n_tiles * c->tile_nsplit)), block(256);
    const size_t sm = gather_smem(c);
    const void *fn = virial ? (c->tile_nsplit > 1 ? (const void *)k_step_small<true, true> : (const void *)k_step_small<true, false>)
                            : (c->tile_nsplit > 1 ? (const void *)k_step_small<false, true> : (const void *)k_step_small<false, false>);
    const cudaError_t e = cudaLaunchCooperativeKernel(fn, grid, block, args, sm, st);
    c->launches++;
    return e != cudaSuccess ? e : cudaGetLastError();
}

TileSums tbsma_tile_sums(const tbsma_ctx *c, double *e_rep, double *ekin, double *w_rep)
{
    TileSums ts;
    ts.cta_sums = c->d_cta_sums;
    ts.tile_first = c->d_tile_first;
    ts.nsplit = use_persist(c) ? c->p_S : c->tile_nsplit;
    ts.e_rep = e_rep; ts.ekin = ekin; ts.w_rep = w_rep;
    return ts;
}

cudaError_t tbsma_launch_reduce_replicas(tbsma_ctx *c, double *e_rep, double *ekin, double *w_rep, cudaStream_t st)
{
    if (!e_rep && !ekin && !w_rep) return cudaSuccess;
    k_reduce_replicas<<<tbsma_reduce_grid(c->R), 256, 0, st>>>(tbsma_tile_sums(c, e_rep, ekin, w_rep), c->R);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_get_neighbors_tile(tbsma_ctx *c, const int32_t *tag, int32_t *counts, int32_t *list,
                                            cudaStream_t st)
{
    k_get_neighbors_tile<<<grid_for(c, c->n, 256, 8), 256, 0, st>>>(tag, reinterpret_cast<const uint2 *>(c->d_nlist),
                                                                   c->d_nn, c->d_tileof, c->d_inv, c->img_cap,
                                                                   c->d_atom_rep, c->d_cur,
                                                                   (size_t)(c->kmax / 4) * c->n_pad, counts, list, (int)c->n,
                                                                   c->n_pad, c->kmax);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_count_pairs_tile(tbsma_ctx *c, const float4 *pos, unsigned long long *d_out2,
                                          cudaStream_t st)
{
    k_count_pairs_tile<<<grid_for(c, c->n, 256, 8), 256, 0, st>>>(pos, reinterpret_cast<const uint2 *>(c->d_nlist),
                                                                 c->d_nn, c->d_tileof, c->d_inv, c->img_cap,
                                                                 c->d_atom_rep, c->d_cur,
                                                                 (size_t)(c->kmax / 4) * c->n_pad, d_out2, (int)c->n, c->n_pad,
                                                                 c->pc.rc2, c->kmax / 4, c->d_geom);
    c->launches++;
    return cudaGetLastError();
}

// what the current lists were built for (bench.py and the tests report it)
extern "C" int tbsma_get_tiling(const tbsma_ctx *c, int32_t *n_tiles, int32_t *box_tiles, int32_t *persistent)
{
    if (!c) return TBSMA_EINVAL;
    const bool tiles = c->active_variant == 2;
    if (n_tiles) *n_tiles = tiles ? c->n_tiles : 0;
    if (box_tiles) *box_tiles = tiles ? c->any_box : 0;
    if (persistent) *persistent = tiles && use_persist(c) ? 1 : 0;
    return TBSMA_OK;
}

// 1 if tbsma_md_run's captured step of the current batch is the single cooperative kernel (tbsma_set_fused_step)
extern "C" int tbsma_get_fused_step(const tbsma_ctx *c)
{
    if (!c) return TBSMA_EINVAL;
    return tbsma_step_small_ok(c) && c->use_graph && c->use_cond ? 1 : 0;
}
