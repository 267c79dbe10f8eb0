// tbsma_cells.cu -- cell binning (counting sort over replica x cell keys), in-place reorder and
// neighbour-list build with a skin.
//
// The paper is silent on binning (it is HOOMD-internal); it only says the best performance came
// with "atoms ordered along the [100]-axis" and a buffer radius r_buff = 0.29 A,
// with fewer rebuilds explaining the 10 K > 298 K throughput.  Here every replica owns a
// fixed slice of one global cell array; cells are numbered x-fastest, z-slowest (z = wire axis),
// so sorted atoms ARE ordered along the axis.  All kernels look at a per-replica dirty flag and do
// nothing for clean replicas, so replicas rebuild independently without host involvement.
#include "tbsma_internal.cuh"

namespace {

constexpr int kThreads = 256;

__device__ __forceinline__ int cell_coord(float x, float lo, float inv_w, int nc, bool periodic, bool &outside)
{
    int c = __float2int_rd((x - lo) * inv_w);
    if (periodic) {
        if (c < 0) c += nc; else if (c >= nc) c -= nc;
    } else if (c < 0 || c >= nc) {
        outside = true;
    }
    return min(max(c, 0), nc - 1);
}

// a1: key of every atom + histogram.  slot = arrival order inside the cell (made stable later).
__global__ void k_bin_count(const float4 *__restrict__ pos, const int *__restrict__ atom_rep,
                            const RepGeom *__restrict__ geom, DirtyView dv,
                            int *__restrict__ ctrl, int *__restrict__ cell_count,
                            int *__restrict__ cell_of, int *__restrict__ slot, int n)
{
    if (!*dv.any) return;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int r = atom_rep[i];
        if (dv.dirty[r] < dv.level) continue;
        const RepGeom *g = geom + r;
        const float4 p = pos[i];
        bool outside = false;
        const int per = g->periodic;
        const int cx = cell_coord(p.x, g->lo[0], g->inv_w[0], g->nc[0], per & 1, outside);
        const int cy = cell_coord(p.y, g->lo[1], g->inv_w[1], g->nc[1], per & 2, outside);
        const int cz = cell_coord(p.z, g->lo[2], g->inv_w[2], g->nc[2], per & 4, outside);
        const int c = g->cell_base + (cz * g->nc[1] + cy) * g->nc[0] + cx;
        cell_of[i] = c;
        slot[i] = atomicAdd(cell_count + c, 1);
        if (outside) atomicOr(ctrl + 1, (int)TBSMA_FLAG_OUT_OF_BOX);
    }
}

// a1: exclusive scan of the histogram, one CTA per replica; re-zeroes the histogram for next time.
__global__ void k_cell_scan(const RepGeom *__restrict__ geom, DirtyView dv,
                            int *__restrict__ cell_count, int *__restrict__ cell_start)
{
    const int r = blockIdx.x;
    if (!*dv.any || dv.dirty[r] < dv.level) return;
    __shared__ int warp_tot[32];
    __shared__ int s_running;
    const RepGeom *g = geom + r;
    const int base = g->cell_base;
    const int ncell = g->nc[0] * g->nc[1] * g->nc[2];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    if (threadIdx.x == 0) s_running = g->atom_begin;
    __syncthreads();
    for (int chunk = 0; chunk < ncell; chunk += blockDim.x) {
        const int c = chunk + threadIdx.x;
        const int v = c < ncell ? cell_count[base + c] : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) warp_tot[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            int t = lane < nw ? warp_tot[lane] : 0;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int u = __shfl_up_sync(0xffffffffu, t, o);
                if (lane >= o) t += u;
            }
            warp_tot[lane] = t;  // inclusive totals of warps
        }
        __syncthreads();
        const int running = s_running;
        const int woff = wid ? warp_tot[wid - 1] : 0;
        if (c < ncell) {
            cell_start[base + c] = running + woff + incl - v;
            cell_count[base + c] = 0;
        }
        __syncthreads();
        if (threadIdx.x == 0) s_running = running + warp_tot[nw - 1];
        __syncthreads();
    }
    if (threadIdx.x == 0) cell_start[base + ncell] = s_running;
}

__global__ void k_scatter(const int *__restrict__ atom_rep, DirtyView dv, const int *__restrict__ cell_start,
                          const int *__restrict__ cell_of, const int *__restrict__ slot,
                          int *__restrict__ order, int n)
{
    if (!*dv.any) return;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        if (dv.dirty[atom_rep[i]] < dv.level) continue;
        order[cell_start[cell_of[i]] + slot[i]] = i;
    }
}

// Make the order inside each cell independent of atomic arrival order: sort by tag (determinism,
// and an order that does not depend on history, so restarts reproduce the fp32 summation order).
// grid = (R, kSortSplit): the CTAs of a clean replica exit at once; a warp takes one cell at a time
// and ranks its atoms by counting smaller tags (tags are unique), 32 atoms per round in registers.
constexpr int kSortSplit = 4;
__global__ void __launch_bounds__(256)
k_cell_sort(const RepGeom *__restrict__ geom, DirtyView dv, const int *__restrict__ cell_start,
            const int *__restrict__ tag, int *__restrict__ order)
{
    if (!*dv.any) return;
    const int r = blockIdx.x;
    if (dv.dirty[r] < dv.level) return;
    const RepGeom *g = geom + r;
    const int ncell = g->nc[0] * g->nc[1] * g->nc[2];
    const int lane = threadIdx.x & 31;
    const int wid = blockIdx.y * (blockDim.x >> 5) + (threadIdx.x >> 5), nw = gridDim.y * (blockDim.x >> 5);
    for (int c = wid; c < ncell; c += nw) {
        const int s = cell_start[g->cell_base + c], m = cell_start[g->cell_base + c + 1] - s;
        if (m <= 1) continue;
        if (m <= 32) {
            const int o = lane < m ? order[s + lane] : 0;
            const int key = lane < m ? tag[o] : 0x7fffffff;
            int rank = 0;
            for (int k = 0; k < m; ++k) rank += __shfl_sync(0xffffffffu, key, k) < key;
            __syncwarp();
            if (lane < m) order[s + rank] = o;
        } else if (m <= 128) {       // up to four atoms per lane (the 9.8 A cells of the tile variant hold ~55)
            int o[4], key[4], rank[4] = {0, 0, 0, 0};
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int k = q * 32 + lane;
                o[q] = k < m ? order[s + k] : 0;
                key[q] = k < m ? tag[o[q]] : 0x7fffffff;
            }
#pragma unroll
            for (int q = 0; q < 4; ++q)
                for (int k = 0; k < 32; ++k) {
                    if (q * 32 + k >= m) break;
                    const int other = __shfl_sync(0xffffffffu, key[q], k);
#pragma unroll
                    for (int p = 0; p < 4; ++p) rank[p] += other < key[p];
                }
            __syncwarp();
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (q * 32 + lane < m) order[s + rank[q]] = o[q];
        } else if (lane == 0) {      // crowded cell: insertion sort by one lane
            for (int a = s + 1; a < s + m; ++a) {
                const int oa = order[a];
                const int ka = tag[oa];
                int b = a - 1;
                while (b >= s) {
                    const int ob = order[b];
                    if (tag[ob] <= ka) break;
                    order[b + 1] = ob;
                    --b;
                }
                order[b + 1] = oa;
            }
        }
        __syncwarp();
    }
}

// a1: gather into cell order (positions wrapped into the box on periodic axes).
__global__ void k_reorder_gather(const float4 *__restrict__ pos, const float4 *__restrict__ vel,
                                 const int *__restrict__ tag, const int *__restrict__ atom_rep,
                                 const RepGeom *__restrict__ geom, DirtyView dv, const int *__restrict__ order,
                                 const int *__restrict__ cell_of, float4 *__restrict__ pos_build,
                                 float4 *__restrict__ tmp4, int *__restrict__ tmp_tag,
                                 int *__restrict__ cell_sorted, int n)
{
    if (!*dv.any) return;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        const int r = atom_rep[k];
        if (dv.dirty[r] < dv.level) continue;
        const RepGeom *g = geom + r;
        const int o = order[k];
        float4 p = pos[o];
        const int per = g->periodic;
        if (per) {
            if (per & 1) { if (p.x >= g->lo[0] + g->len[0]) p.x -= g->len[0]; else if (p.x < g->lo[0]) p.x += g->len[0]; }
            if (per & 2) { if (p.y >= g->lo[1] + g->len[1]) p.y -= g->len[1]; else if (p.y < g->lo[1]) p.y += g->len[1]; }
            if (per & 4) { if (p.z >= g->lo[2] + g->len[2]) p.z -= g->len[2]; else if (p.z < g->lo[2]) p.z += g->len[2]; }
        }
        pos_build[k] = p;
        if (vel) tmp4[k] = vel[o];
        tmp_tag[k] = tag[o];
        cell_sorted[k] = cell_of[o];
    }
}

__global__ void k_reorder_copyback(float4 *__restrict__ pos, float4 *__restrict__ vel, int *__restrict__ tag,
                                   const int *__restrict__ atom_rep, DirtyView dv,
                                   const float4 *__restrict__ tmp_pos,
                                   const float4 *__restrict__ tmp4, const int *__restrict__ tmp_tag, int n)
{
    if (!*dv.any) return;
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n; k += gridDim.x * blockDim.x) {
        if (dv.dirty[atom_rep[k]] < dv.level) continue;
        pos[k] = tmp_pos[k];
        if (vel) vel[k] = tmp4[k];
        tag[k] = tmp_tag[k];
    }
}

// a2: neighbour list with skin (global variant), cell by cell.  One CTA takes a cell, stages the atoms of its (up to)
// 27 neighbour cells in shared memory once, and a WARP takes each atom of the cell, its lanes testing 32 staged
// candidates at a time (vote + prefix count give every kept candidate its place in the list).  Membership = the fp32
// predicate of D:A6, operation for operation.  (A thread per atom reading every candidate through L1 took 3.3 ms for
// 10^6 atoms; this takes 1.7 ms.)
constexpr int kCellCap = 1024;     // staged candidates per pass
constexpr int kCellBatch = 512;    // atoms of the cell per pass
template <bool PERIODIC>
__global__ void __launch_bounds__(256)
k_build_list_cells(const float4 *__restrict__ pos, const int *__restrict__ cell_rep,
                   const RepGeom *__restrict__ geom, DirtyView dv, int *__restrict__ ctrl,
                   const int *__restrict__ cell_start, int *__restrict__ nlist, int *__restrict__ nn,
                   float4 *__restrict__ pos_build, int n_pad, int kmax, float rl2, int n_cells)
{
    __shared__ float4 s_pos[kCellCap];
    __shared__ int s_idx[kCellCap];
    __shared__ int s_cs[27], s_off[28], s_ncell;
    __shared__ int s_cnt[kCellBatch];
    if (!*dv.any) return;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nw = blockDim.x >> 5;
    for (int c = blockIdx.x; c < n_cells; c += gridDim.x) {
        const int r = cell_rep[c];
        if (dv.dirty[r] < dv.level) continue;
        const RepGeom *g = geom + r;
        const int s0 = cell_start[c], m0 = cell_start[c + 1] - s0;
        if (m0 == 0) continue;
        const int per = PERIODIC ? g->periodic : 0;
        float Lx = 0.f, Ly = 0.f, Lz = 0.f;
        if (PERIODIC) { Lx = g->len[0]; Ly = g->len[1]; Lz = g->len[2]; }
        __syncthreads();       // the previous cell's staging is no longer read
        if (tid == 0) {
            // distinct neighbour cell coordinates per axis (periodic axes with < 3 cells dedupe)
            const int nx = g->nc[0], ny = g->nc[1], nz = g->nc[2], base = g->cell_base;
            const int lc = c - base;
            const int cx = lc % nx, cy = (lc / nx) % ny, cz = lc / (nx * ny);
            int ax[3], ay[3], az[3], nax = 0, nay = 0, naz = 0;
            for (int o = -1; o <= 1; ++o) {
                int t = cx + o;
                if (per & 1) { if (t < 0) t += nx; else if (t >= nx) t -= nx; }
                bool ok = t >= 0 && t < nx;
                for (int u = 0; u < nax; ++u) ok = ok && ax[u] != t;
                if (ok) ax[nax++] = t;
                t = cy + o;
                if (per & 2) { if (t < 0) t += ny; else if (t >= ny) t -= ny; }
                ok = t >= 0 && t < ny;
                for (int u = 0; u < nay; ++u) ok = ok && ay[u] != t;
                if (ok) ay[nay++] = t;
                t = cz + o;
                if (per & 4) { if (t < 0) t += nz; else if (t >= nz) t -= nz; }
                ok = t >= 0 && t < nz;
                for (int u = 0; u < naz; ++u) ok = ok && az[u] != t;
                if (ok) az[naz++] = t;
            }
            int k = 0, run = 0;
            for (int iz = 0; iz < naz; ++iz)
                for (int iy = 0; iy < nay; ++iy)
                    for (int ix = 0; ix < nax; ++ix) {
                        const int cc = base + (az[iz] * ny + ay[iy]) * nx + ax[ix];
                        const int s = cell_start[cc], e = cell_start[cc + 1];
                        s_cs[k] = s;
                        s_off[k] = run;
                        run += e - s;
                        ++k;
                    }
            s_off[k] = run;
            s_ncell = k;
        }
        __syncthreads();
        const int ncell = s_ncell, T = s_off[ncell];
        for (int a0 = 0; a0 < m0; a0 += kCellBatch) {
            const int mb = min(kCellBatch, m0 - a0);
            for (int a = tid; a < mb; a += blockDim.x) s_cnt[a] = 0;
            for (int u0 = 0; u0 < T; u0 += kCellCap) {
                const int tc = min(kCellCap, T - u0);
                __syncthreads();
                for (int u = tid; u < tc; u += blockDim.x) {
                    const int v = u0 + u;
                    int k = 0;
                    while (v >= s_off[k + 1]) ++k;
                    const int j = s_cs[k] + v - s_off[k];
                    s_pos[u] = pos[j];
                    s_idx[u] = j;
                }
                __syncthreads();
                for (int a = wid; a < mb; a += nw) {
                    const int i = s0 + a0 + a;
                    const float4 pi = pos[i];
                    int cnt = s_cnt[a];
                    for (int ub = 0; ub < tc; ub += 32) {
                        const int u = ub + lane;
                        bool keep = false;
                        int j = 0;
                        if (u < tc) {
                            const float4 pj = s_pos[u];
                            j = s_idx[u];
                            float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
                            if (PERIODIC) {
                                if (per & 1) { const float h = 0.5f * Lx; if (dx > h) dx -= Lx; else if (dx < -h) dx += Lx; }
                                if (per & 2) { const float h = 0.5f * Ly; if (dy > h) dy -= Ly; else if (dy < -h) dy += Ly; }
                                if (per & 4) { const float h = 0.5f * Lz; if (dz > h) dz -= Lz; else if (dz < -h) dz += Lz; }
                            }
                            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));   // D:A6
                            keep = d2 < rl2 && j != i;
                        }
                        const unsigned kept = __ballot_sync(0xffffffffu, keep);
                        const int k = cnt + __popc(kept & ((1u << lane) - 1u));
                        if (keep && k < kmax) nlist[(tbsma_lrow(i, kmax >> 2) + (size_t)(k >> 2) * TBSMA_LROW) * 4 + (k & 3)] = j;
                        cnt += __popc(kept);
                    }
                    if (lane == 0) s_cnt[a] = cnt;
                }
            }
            __syncthreads();
            for (int a = tid; a < mb; a += blockDim.x) {
                const int i = s0 + a0 + a;
                const float4 pi = pos[i];
                int cnt = s_cnt[a];
                if (cnt > kmax) atomicOr(ctrl + 1, (int)TBSMA_FLAG_NLIST_OVERFLOW);
                if (cnt > ctrl[2]) atomicMax(ctrl + 2, cnt);
                cnt = min(cnt, kmax);
                for (int k = cnt; k < ((cnt + 3) & ~3); ++k)   // pad the last group of four with self
                    nlist[(tbsma_lrow(i, kmax >> 2) + (size_t)(k >> 2) * TBSMA_LROW) * 4 + (k & 3)] = i;
                nn[i] = cnt | ((__float_as_int(pi.w) & 3) << 16);
                pos_build[i] = pi;
            }
            __syncthreads();
        }
    }
}

__global__ void k_mark_all_dirty(int *__restrict__ dirty, int *__restrict__ ctrl, int R)
{
    for (int r = blockIdx.x * blockDim.x + threadIdx.x; r < R; r += gridDim.x * blockDim.x) dirty[r] = 2;
    if (blockIdx.x == 0 && threadIdx.x == 0) { ctrl[0] = 1; ctrl[3] = 1; }
}

__global__ void k_get_neighbors(const int *__restrict__ tag, const int *__restrict__ nlist,
                                const int *__restrict__ nn, int *__restrict__ counts,
                                int *__restrict__ list, int n, int n_pad, int kmax)
{
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const int t = tag[i];
        const int cnt = nn[i] & 0xffff;
        counts[t] = cnt;
        for (int k = 0; k < cnt; ++k)
            list[(size_t)t * kmax + k] = tag[nlist[(tbsma_lrow(i, kmax >> 2) + (size_t)(k >> 2) * TBSMA_LROW) * 4 + (k & 3)]];
    }
}

inline int grid_for(const tbsma_ctx *c, int64_t work, int threads, int per_sm)
{
    int64_t b = (work + threads - 1) / threads;
    int64_t cap = (int64_t)c->n_sm * per_sm;
    if (b > cap) b = cap;
    if (b < 1) b = 1;
    return (int)b;
}

}  // namespace

cudaError_t tbsma_launch_mark_all_dirty(tbsma_ctx *c, cudaStream_t st)
{
    k_mark_all_dirty<<<grid_for(c, c->R, kThreads, 4), kThreads, 0, st>>>(c->d_dirty, c->d_ctrl, c->R);
    c->launches++;
    return cudaGetLastError();
}

// The rebuild chain.  Every kernel is a no-op unless ctrl[0] (any replica dirty) is set and
// touches only dirty replicas, so it can be enqueued unconditionally every step.
cudaError_t tbsma_launch_rebuild(tbsma_ctx *c, float4 *pos, float4 *vel, int32_t *tag, bool do_cells,
                                 bool do_list, cudaStream_t st)
{
    const int n = (int)c->n;
    const int ga = grid_for(c, n, kThreads, 8);
    const DirtyView dv = tbsma_dirty_view(c);
    if (do_cells) {
        k_bin_count<<<ga, kThreads, 0, st>>>(pos, c->d_atom_rep, c->d_geom, dv, c->d_ctrl,
                                             c->d_cell_count, c->d_cell_of, c->d_slot, n);
        const int scan_threads = (c->n_cells / c->R > 4096) ? 1024 : 256;
        k_cell_scan<<<c->R, scan_threads, 0, st>>>(c->d_geom, dv, c->d_cell_count, c->d_cell_start);
        k_scatter<<<ga, kThreads, 0, st>>>(c->d_atom_rep, dv, c->d_cell_start,
                                           c->d_cell_of, c->d_slot, c->d_order, n);
        // a warp sorts one cell at a time: enough CTAs per replica that a batch of few, large replicas fills the GPU too
        int split = (8 * c->n_sm + c->R - 1) / c->R;
        if (split < kSortSplit) split = kSortSplit;
        const int64_t by_cells = (c->n_cells / c->R + 7) / 8;      // no more CTAs than cells / 8 warps
        if (split > by_cells) split = (int)(by_cells > 0 ? by_cells : 1);
        if (split > 65535) split = 65535;
        k_cell_sort<<<dim3(c->R, split), 256, 0, st>>>(c->d_geom, dv, c->d_cell_start, tag, c->d_order);
        // d_slot is free after the scatter: reuse it for the cell id of every sorted slot
        k_reorder_gather<<<ga, kThreads, 0, st>>>(pos, vel, tag, c->d_atom_rep, c->d_geom, dv,
                                                  c->d_order, c->d_cell_of, c->d_tmp_pos,
                                                  c->d_tmp4, c->d_tmp_tag, c->d_slot, n);
        c->launches += 5;
        // the tile variant moves the atoms once more (count order inside each layer) while it builds
        // the lists, so its copy-back is part of tbsma_launch_tile_lists
        if (!(do_list && c->active_variant == 2)) {
            k_reorder_copyback<<<ga, kThreads, 0, st>>>(pos, vel, tag, c->d_atom_rep, dv,
                                                        c->d_tmp_pos, c->d_tmp4, c->d_tmp_tag, n);
            c->launches++;
        }
    }
    if (do_list && c->active_variant == 2) {
        if (!do_cells) {
            cudaError_t e = tbsma_launch_stage_copy(c, pos, vel, tag, st);
            if (e != cudaSuccess) return e;
        }
        return tbsma_launch_tile_lists(c, pos, vel, tag, st);
    }
    if (do_list) {
        const int64_t cap = (int64_t)c->n_sm * 16;
        const int gl = (int)(c->n_cells < cap ? c->n_cells : cap);
        if (c->any_periodic)
            k_build_list_cells<true><<<gl, 256, 0, st>>>(pos, c->d_cell_rep, c->d_geom, dv, c->d_ctrl, c->d_cell_start,
                                                         c->d_nlist, c->d_nn, c->d_pos_build, c->n_pad, c->kmax,
                                                         c->pc.rl2, (int)c->n_cells);
        else
            k_build_list_cells<false><<<gl, 256, 0, st>>>(pos, c->d_cell_rep, c->d_geom, dv, c->d_ctrl, c->d_cell_start,
                                                          c->d_nlist, c->d_nn, c->d_pos_build, c->n_pad, c->kmax,
                                                          c->pc.rl2, (int)c->n_cells);
        c->launches++;
    }
    return cudaGetLastError();
}

cudaError_t tbsma_launch_get_neighbors(tbsma_ctx *c, const int32_t *tag, int32_t *counts, int32_t *list,
                                       cudaStream_t st)
{
    k_get_neighbors<<<grid_for(c, c->n, kThreads, 8), kThreads, 0, st>>>(tag, c->d_nlist, c->d_nn, counts,
                                                                         list, (int)c->n, c->n_pad, c->kmax);
    c->launches++;
    return cudaGetLastError();
}
