// tbsma_api.cu -- the C ABI declared in include/tbsma.h: argument checking, host-side geometry,
// scratch ownership and the launch sequences.  No arithmetic of the method lives here.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "tbsma_internal.cuh"

#define CK(call)                                   \
    do {                                           \
        cudaError_t e_ = (call);                   \
        if (e_ != cudaSuccess) return map_cuda(e_); \
    } while (0)

namespace {

int map_cuda(cudaError_t e)
{
    if (e == cudaErrorMemoryAllocation) return TBSMA_ENOMEM;
    return TBSMA_ECUDA;
}

template <class T>
cudaError_t dalloc(T **p, size_t count)
{
    *p = nullptr;
    if (count == 0) count = 1;
    return cudaMalloc((void **)p, count * sizeof(T));
}

void free_system(tbsma_ctx *c)
{
    cudaFree(c->d_geom); cudaFree(c->d_atom_rep); cudaFree(c->d_cell_count); cudaFree(c->d_cell_start);
    cudaFree(c->d_cell_rep); c->d_cell_rep = nullptr;
    cudaFree(c->d_cell_of); cudaFree(c->d_slot); cudaFree(c->d_order); cudaFree(c->d_pos_build);
    cudaFree(c->d_tmp4); cudaFree(c->d_tmp_tag); cudaFree(c->d_nlist); cudaFree(c->d_nn); cudaFree(c->d_xs);
    cudaFree(c->d_dirty); cudaFree(c->d_ctrl); cudaFree(c->d_counters); cudaFree(c->d_stagger); cudaFree(c->d_cur);
    cudaFree(c->d_nh); cudaFree(c->d_kmid); cudaFree(c->d_nh_scale); cudaFree(c->d_blk_rep); cudaFree(c->d_blk_first);
    c->d_stagger = nullptr; c->d_cur = nullptr; c->d_nh = nullptr; c->d_kmid = nullptr; c->d_nh_scale = nullptr;
    c->d_blk_rep = nullptr; c->d_blk_first = nullptr; c->n_blk = 0;
    cudaFree(c->d_tiles); cudaFree(c->d_maxpop); cudaFree(c->d_hbase); cudaFree(c->d_tileof); cudaFree(c->d_img); cudaFree(c->d_inv);
    c->d_tileof = nullptr; c->d_img = nullptr; c->d_inv = nullptr;
    cudaFree(c->d_cta_sums); c->d_cta_sums = nullptr; c->have_sums = 0;
    cudaFree(c->d_series_w); c->d_series_w = nullptr;
    memset(&c->series, 0, sizeof(c->series));
    cudaFree(c->d_newslot); cudaFree(c->d_oldof);
    cudaFree(c->d_nn_tmp); cudaFree(c->d_tmp_pos);
    cudaFree(c->d_tile_first); cudaFree(c->d_work);
    c->d_tile_first = nullptr; c->d_work = nullptr;
    cudaFree(c->d_olist); cudaFree(c->d_nn_o); cudaFree(c->d_pos_outer); cudaFree(c->d_want_outer);
    c->d_olist = nullptr; c->d_nn_o = nullptr; c->d_pos_outer = nullptr; c->d_want_outer = nullptr;
    c->d_tiles = nullptr; c->d_maxpop = nullptr; c->d_hbase = nullptr; c->d_newslot = nullptr; c->d_oldof = nullptr;
    c->d_nn_tmp = nullptr; c->d_tmp_pos = nullptr;
    c->n_tiles = 0; c->active_variant = 1;
    c->d_geom = nullptr; c->d_atom_rep = nullptr; c->d_cell_count = nullptr; c->d_cell_start = nullptr;
    c->d_cell_of = nullptr; c->d_slot = nullptr; c->d_order = nullptr; c->d_pos_build = nullptr;
    c->d_tmp4 = nullptr; c->d_tmp_tag = nullptr; c->d_nlist = nullptr; c->d_nn = nullptr; c->d_xs = nullptr;
    c->d_dirty = nullptr; c->d_ctrl = nullptr; c->d_counters = nullptr;
    free(c->h_off); free(c->h_geom);
    c->h_off = nullptr; c->h_geom = nullptr;
    c->cells_built = c->list_built = 0;
}

void free_staging(tbsma_ctx *c)
{
    cudaFree(c->s_pos); cudaFree(c->s_vel); cudaFree(c->s_force); cudaFree(c->s_tag); cudaFree(c->s_T);
    cudaFree(c->s_seed); cudaFree(c->s_disp0); cudaFree(c->s_rate); cudaFree(c->s_e); cudaFree(c->s_w); cudaFree(c->s_k);
    c->s_pos = c->s_vel = c->s_force = nullptr; c->s_tag = nullptr; c->s_T = nullptr; c->s_seed = nullptr;
    c->s_disp0 = c->s_rate = c->s_e = c->s_w = c->s_k = nullptr;
    c->s_n = 0; c->s_R = 0;
}

// Fold the pair-function constants in double, round once to fp32.
void fold_constants(tbsma_ctx *c)
{
    const tbsma_params &P = c->prm;
    PairConst &k = c->pc;
    const float rc = (float)c->r_cut, rl = (float)(c->r_cut + c->skin);
    k.rc2 = rc * rc;   // fp32 product, as D:A6 prescribes
    k.rl2 = rl * rl;
    const float ro = (float)(c->r_cut + c->skin + c->outer_skin);
    k.ro2 = ro * ro;
    k.r0f = (float)P.r0;
    const double log2e = 1.4426950408889634074;
    const double aq = -2.0 * P.q / P.r0 * log2e, ap = -P.p / P.r0 * log2e;
    const double dr0 = (double)k.r0f - P.r0;     // t = r - r0f  =>  r - r0 = t + dr0
    k.aq = (float)aq;
    k.ap = (float)ap;
    k.b_rho = (float)(log2(P.xi * P.xi) + aq * dr0);
    k.b_rep = (float)(log2(2.0 * P.A * P.p / P.r0) + ap * dr0);
    k.b_band = (float)(log2(P.q * P.xi * P.xi / P.r0) + aq * dr0);
    k.e_rep_scale = (float)(P.r0 / (2.0 * P.p));
}


// Cell grid of every replica for cells at least `width` wide (+ a margin over the fp32 rounding of cell
// coordinates); (re)allocates the cell arrays.  The tile variant scans for candidates within
// r_cut + skin + outer_skin, the global variant for list members within r_cut + skin.
int set_geometry(tbsma_ctx *c, double width)
{
    const int R = c->R;
    const double w_min = width * (1.0 + 1e-5) + 1e-4;
    int64_t cells = 0;
    for (int r = 0; r < R; ++r) {
        RepGeom &g = c->h_geom[r];
        int64_t nc_r = 1;
        for (int a = 0; a < 3; ++a) {
            const float len = g.len[a];
            int nc = (int)floor((double)len / w_min);
            if (nc < 1) nc = 1;
            if (nc > 1024) nc = 1024;
            g.nc[a] = nc;
            g.inv_w[a] = len > 0.0f ? (float)((double)nc / (double)len) : 0.0f;
            nc_r *= nc;
        }
        g.cell_base = (int)cells;
        cells += nc_r;
        if (cells > 0x7ffffff0ll) return TBSMA_EINVAL;
    }
    cudaFree(c->d_cell_count); cudaFree(c->d_cell_start); cudaFree(c->d_cell_rep);
    c->d_cell_count = nullptr; c->d_cell_start = nullptr; c->d_cell_rep = nullptr;
    c->n_cells = cells;
    c->cell_w = width;
    CK(dalloc(&c->d_cell_count, (size_t)cells));
    CK(dalloc(&c->d_cell_rep, (size_t)cells));
    {
        int32_t *h = (int32_t *)malloc(sizeof(int32_t) * (size_t)(cells ? cells : 1));
        if (!h) return TBSMA_ENOMEM;
        for (int r = 0; r < R; ++r) {
            const RepGeom &g = c->h_geom[r];
            const int64_t nc_r = (int64_t)g.nc[0] * g.nc[1] * g.nc[2];
            for (int64_t k = 0; k < nc_r; ++k) h[g.cell_base + k] = r;
        }
        const cudaError_t ce = cudaMemcpy(c->d_cell_rep, h, sizeof(int32_t) * (size_t)cells, cudaMemcpyHostToDevice);
        free(h);
        CK(ce);
    }
    CK(dalloc(&c->d_cell_start, (size_t)cells + 1));
    CK(cudaMemset(c->d_cell_count, 0, sizeof(int32_t) * (size_t)cells));
    CK(cudaMemset(c->d_cell_start, 0, sizeof(int32_t) * ((size_t)cells + 1)));
    CK(cudaMemcpy(c->d_geom, c->h_geom, sizeof(RepGeom) * R, cudaMemcpyHostToDevice));
    return TBSMA_OK;
}

// The shared-memory tile variant cuts a periodic replica into boxes of cells with a one-cell halo that must not wrap onto
// itself: at least three cells (of the candidate radius) along every periodic axis.  Shorter periodic boxes use the global
// variant with its own, narrower cells.
bool tiles_possible(const tbsma_ctx *c)
{
    if (c->variant == 1 || (c->variant == 0 && c->tiles_rejected)) return false;
    const double w_min = (c->r_cut + c->skin + c->outer_skin) * (1.0 + 1e-5) + 1e-4;
    for (int r = 0; r < c->R; ++r)
        for (int a = 0; a < 3; ++a)
            if ((c->h_geom[r].periodic >> a & 1) && (int)floor((double)c->h_geom[r].len[a] / w_min) < 3) return false;
    return true;
}

// Cell width and candidate-list storage for the variant the next build will try (called by tbsma_build_cells).
int ensure_variant_resources(tbsma_ctx *c)
{
    const bool tiles = tiles_possible(c);
    const double r_list = c->r_cut + c->skin;
    const double width = tiles ? r_list + c->outer_skin : r_list;
    if (width != c->cell_w) {
        CK(cudaDeviceSynchronize());
        const int rc = set_geometry(c, width);
        if (rc) return rc;
    }
    if (tiles && !c->d_olist) {
        const double ratio = (r_list + c->outer_skin) / r_list;
        int ko = (int)ceil(c->kmax * ratio * ratio * ratio * 1.25) + 8;   // volume ratio + room for a lattice shell
        ko = (ko + 3) / 4 * 4;
        if (ko > 248) ko = 248;        // byte-packed class counters of k_tile_finish
        if (ko < c->kmax) ko = c->kmax;
        c->kmax_o = ko;
        const size_t n = (size_t)c->n;
        CK(dalloc(&c->d_olist, (size_t)2 * (ko / 4) * (size_t)c->n_pad));
        CK(dalloc(&c->d_nn_o, n));
        CK(dalloc(&c->d_pos_outer, n));
        CK(dalloc(&c->d_want_outer, (size_t)c->R));
        CK(cudaMemset(c->d_want_outer, 0, sizeof(int32_t) * (size_t)c->R));
        CK(cudaMemset(c->d_nn_o, 0, sizeof(int32_t) * (n ? n : 1)));
    }
    return TBSMA_OK;
}

int run_steps(tbsma_ctx *c, float4 *pos, float4 *vel, float4 *force, int32_t *tag, double dt, const float *T,
              double gamma, const unsigned long long *seed, unsigned long long step0, int64_t n_steps,
              const double *disp0, const double *rate, int rebuild_every, double *e_rep, double *w_rep,
              double *ekin, bool advance, cudaStream_t st, bool step_on_device = false)
{
    StepArgs a;
    a.step_on_device = step_on_device ? 1 : 0;
    a.half_dt = (float)(0.5 * dt);
    a.kick = (float)(0.5 * dt * TBSMA_ACC / c->prm.mass_amu);
    const double c1 = exp(-gamma * dt);
    a.c1 = (float)c1;
    a.c2 = (float)sqrt(1.0 - c1 * c1);
    a.sigma_scale = (float)sqrt(TBSMA_KB * TBSMA_ACC / c->prm.mass_amu);
    a.skin_half2 = (float)(0.25 * c->skin * c->skin);
    a.trigger2 = a.skin_half2;
    const bool tiles = c->active_variant == 2;
    const bool async = tiles && c->async_inner && c->list_bufs == 2 && rebuild_every <= 0 &&
                       0.5 * c->skin > c->async_margin && c->async_margin > 0.0;
    if (async) a.trigger2 = (float)((0.5 * c->skin - c->async_margin) * (0.5 * c->skin - c->async_margin));
    a.cur = c->d_cur;
    a.pb_stride = c->n_pad;
    const bool nose_hoover = c->thermostat_kind == 1;
    a.thermostat = !nose_hoover && gamma > 0.0;
    a.nh_scale = nose_hoover ? c->d_nh_scale : nullptr;
    a.rebuild_every = rebuild_every;
    a.step_base = step0;
    a.T = T; a.seed = seed; a.disp0 = disp0; a.rate = rate;
    a.want_outer = c->active_variant == 2 ? c->d_want_outer : nullptr;
    a.stagger = c->d_stagger;
    a.disp0_1 = c->proto.d_slab1_disp0; a.rate_1 = c->proto.d_slab1_rate;
    a.period = (long long)c->proto.stepwise_period;
    a.T_rate = c->proto.d_T_rate;
    // a series of the tensile observables needs the virial of every step it records
    const bool series = advance && c->series.every > 0 && c->series.d_series;
    if (series && !w_rep) w_rep = c->d_series_w;
    a.e_rep = e_rep; a.w_rep = w_rep; a.ekin = ekin;
    KickArgs kk;
    kk.vel = vel; kk.kick = a.kick; kk.ke_scale = (float)(0.5 * c->prm.mass_amu / TBSMA_ACC); kk.ekin = ekin;
    for (int64_t s = 0; s < n_steps; ++s) {
        cudaEvent_t *ev = nullptr;
        if (c->timing && c->tev && c->tev_steps < TBSMA_TIMING_MAX_STEPS) ev = c->tev + 6 * (c->tev_steps++);
        if (ev) CK(cudaEventRecord(ev[0], st));
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        cudaGraph_t cg = nullptr;
        const cudaGraphNode_t *deps = nullptr;
        size_t n_deps = 0;
        cudaGraphConditionalHandle cond = 0;
        bool use_cond = false;
        if (tiles) {
            if (st && c->use_cond && c->body_stream &&
                cudaStreamGetCaptureInfo(st, &cap, nullptr, &cg, &deps, &n_deps) == cudaSuccess &&
                cap == cudaStreamCaptureStatusActive && cg)
                use_cond = cudaGraphConditionalHandleCreate(&cond, cg, 0, cudaGraphCondAssignDefault) == cudaSuccess;
        }
        if (nose_hoover) CK(tbsma_launch_nose_hoover(c, pos, vel, force, a, dt, st));
        if (tiles && use_cond && !ev && tbsma_step_small_ok(c)) {
            // Small batch: the whole step is ONE cooperative kernel (k_step_small).  Only when the displacement check in it
            // finds a replica that needs a new list is the rest of the step run by the ordinary kernels, the body of an IF.
            const int sync_level_f = async ? 2 : 1;
            CK(tbsma_launch_step_small(c, pos, vel, force, tag, a, kk, w_rep != nullptr, (advance ? 1 : 0) | 2,
                                       tbsma_tile_sums(c, e_rep, ekin, w_rep), (unsigned long long)cond, st));
            CK(cudaStreamGetCaptureInfo(st, &cap, nullptr, &cg, &deps, &n_deps));
            cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
            np.type = cudaGraphNodeTypeConditional;
            np.conditional.handle = cond;
            np.conditional.type = cudaGraphCondTypeIf;
            np.conditional.size = 1;
            cudaGraphNode_t cnode;
            CK(cudaGraphAddNode(&cnode, cg, deps, n_deps, &np));
            cudaGraph_t body = np.conditional.phGraph_out[0];
            cudaStream_t bs = c->body_stream;
            CK(cudaStreamBeginCaptureToGraph(bs, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
            const int64_t before = c->launches;
            cudaError_t eb = tbsma_launch_tile_worklist(c, bs, 0ull, 0);
            if (eb == cudaSuccess) eb = tbsma_launch_rebuild(c, pos, vel, tag, true, true, bs);
            if (eb == cudaSuccess) eb = tbsma_launch_tile_inner(c, pos, 1, bs);
            if (eb == cudaSuccess) eb = tbsma_launch_tile_inner(c, pos, 0, bs);
            if (eb == cudaSuccess) eb = tbsma_launch_density_tile(c, pos, sync_level_f, bs, false);
            if (eb == cudaSuccess) eb = tbsma_launch_force_tile(c, force, w_rep != nullptr, kk, sync_level_f, bs);
            if (eb == cudaSuccess) eb = tbsma_launch_finish_step(c, (advance ? 1 : 0) | 2, bs, tbsma_tile_sums(c, e_rep, ekin, w_rep));
            c->launches = before;      // (the body runs in the few steps that renew a list)
            cudaGraph_t body_out = nullptr;
            CK(cudaStreamEndCapture(bs, &body_out));
            CK(eb);
            CK(cudaStreamUpdateCaptureDependencies(st, &cnode, 1, cudaStreamSetCaptureDependencies));
            if (series) CK(tbsma_launch_series_record(c, pos, vel, w_rep, a, st));
            continue;
        }
        CK(tbsma_launch_integrate_pre(c, pos, vel, force, tag, a, st));
        if (ev) CK(cudaEventRecord(ev[1], st));
        bool forked = false, early = false, joined = false;
        if (tiles) {
            // Replicas whose atoms moved far enough get a new list.  With new cells and candidates (dirty == 2, rare)
            // the rebuild precedes the gather passes, which then read the freshly written half of the list buffers.
            // A list that is only re-filtered from its candidates (dirty == 1) is, when `async`, asked for `margin`
            // early and written to the other half while the gather passes of this step still read the old one, on a
            // second stream; the step's last kernel swaps the halves.
            CK(tbsma_launch_tile_worklist(c, st, (unsigned long long)cond, use_cond ? 1 : 0));
            if (use_cond) {
                // IF (a replica needs new cells and candidates) { chain; its inner lists }: nothing is launched otherwise
                CK(cudaStreamGetCaptureInfo(st, &cap, nullptr, &cg, &deps, &n_deps));
                cudaGraphNodeParams np = {cudaGraphNodeTypeConditional};
                np.type = cudaGraphNodeTypeConditional;
                np.conditional.handle = cond;
                np.conditional.type = cudaGraphCondTypeIf;
                np.conditional.size = 1;
                cudaGraphNode_t cnode;
                CK(cudaGraphAddNode(&cnode, cg, deps, n_deps, &np));
                cudaGraph_t body = np.conditional.phGraph_out[0];
                CK(cudaStreamBeginCaptureToGraph(c->body_stream, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
                const int64_t before = c->launches;
                cudaError_t e1 = tbsma_launch_rebuild(c, pos, vel, tag, true, true, c->body_stream);
                cudaError_t e2 = tbsma_launch_tile_inner(c, pos, 1, c->body_stream);
                c->launches = before;      // kernels of the body are not counted: they run in a few steps only
                cudaGraph_t body_out = nullptr;
                CK(cudaStreamEndCapture(c->body_stream, &body_out));
                CK(e1);
                CK(e2);
                CK(cudaStreamUpdateCaptureDependencies(st, &cnode, 1, cudaStreamSetCaptureDependencies));
            } else {
                CK(tbsma_launch_rebuild(c, pos, vel, tag, true, true, st));
                CK(tbsma_launch_tile_inner(c, pos, 1, st));
            }
            // (after the chain: idle, its kernels take 1.5 us each on an empty GPU, but each would wait for room on every SM
            // behind a filter kernel already running)
            if (async && c->overlap == 2 && !c->timing && st) {
                CK(tbsma_launch_tile_inner(c, pos, 0, st, true));
                early = true;
                forked = true;       // (nothing to join: same stream)
                joined = true;
            } else if (async && c->overlap && !c->timing && c->aux_stream) {
                CK(cudaEventRecord(c->ev_fork, st));
                CK(cudaStreamWaitEvent(c->aux_stream, c->ev_fork, 0));
                CK(tbsma_launch_tile_inner(c, pos, 0, c->aux_stream, true));
                CK(cudaEventRecord(c->ev_join, c->aux_stream));
                forked = true;
            }
            if (!forked) CK(tbsma_launch_tile_inner(c, pos, 0, st));
        } else {
            CK(tbsma_launch_rebuild(c, pos, vel, tag, true, true, st));
        }
        const int sync_level = async ? 2 : 1;
        if (ev) CK(cudaEventRecord(ev[2], st));
        if (tiles) CK(tbsma_launch_density_tile(c, pos, sync_level, st, early));
        else CK(tbsma_launch_density(c, pos, st));
        if (ev) CK(cudaEventRecord(ev[3], st));
        if (tiles) CK(tbsma_launch_force_tile(c, force, w_rep != nullptr, kk, sync_level, st));
        else CK(tbsma_launch_force(c, force, e_rep, w_rep, kk, st));
        if (ev) CK(cudaEventRecord(ev[4], st));
        if (forked && !joined) CK(cudaStreamWaitEvent(st, c->ev_join, 0));
        CK(tbsma_launch_finish_step(c, (advance ? 1 : 0) | 2, st,
                                    tiles ? tbsma_tile_sums(c, e_rep, ekin, w_rep) : TileSums()));
        if (series) CK(tbsma_launch_series_record(c, pos, vel, w_rep, a, st));
        if (ev) CK(cudaEventRecord(ev[5], st));
    }
    return TBSMA_OK;
}

}  // namespace

extern "C" {

const char *tbsma_version(void) { return "tbsma-b200 0.1 (sm_100a)"; }

const char *tbsma_strerror(int code)
{
    switch (code) {
        case TBSMA_OK: return "ok";
        case TBSMA_EINVAL: return "invalid argument";
        case TBSMA_ENOMEM: return "out of memory";
        case TBSMA_ECUDA: return "CUDA runtime error (or no CUDA device)";
        case TBSMA_ESTATE: return "call order violated";
        case TBSMA_ELIMIT: return "size exceeds the fixed capacity of a no-allocation entry point";
        default: return "unknown error";
    }
}

int tbsma_create(const tbsma_params *params, double r_cut, double skin, tbsma_ctx **out)
{
    if (!params || !out || !(r_cut > 0.0) || !(skin >= 0.0) || !(params->r0 > 0.0) || !(params->mass_amu > 0.0) ||
        !(params->xi > 0.0) || !(params->A > 0.0))
        return TBSMA_EINVAL;
    *out = nullptr;
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return TBSMA_ECUDA;   // no CPU fallback
    CK(cudaGetDevice(&dev));
    tbsma_ctx *c = (tbsma_ctx *)calloc(1, sizeof(tbsma_ctx));
    if (!c) return TBSMA_ENOMEM;
    c->prm = *params;
    c->r_cut = r_cut;
    c->skin = skin;
    c->device = dev;
    c->variant = 0;
    c->active_variant = 1;
    c->outer_skin = 2.5;
    c->tile_layers = 2;
    c->tile_threads = 256;
    c->gather_mode = 1;
    c->fused_step = 1;
    c->use_graph = 1;
    c->overlap = 2;
    c->stagger = 1;
    c->balance = 1;
    c->class_h = params->r0 / sqrt(2.0);
    c->use_cond = 1;
    c->async_inner = 1;
    c->async_margin = 0.03;
    {
        int lo_prio = 0, hi_prio = 0;
        cudaDeviceGetStreamPriorityRange(&lo_prio, &hi_prio);
        if (cudaStreamCreateWithPriority(&c->aux_stream, cudaStreamNonBlocking, hi_prio) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming) != cudaSuccess) {
            if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
            if (c->ev_fork) cudaEventDestroy(c->ev_fork);
            free(c);
            return TBSMA_ECUDA;
        }
        if (cudaStreamCreateWithFlags(&c->body_stream, cudaStreamNonBlocking) != cudaSuccess) c->body_stream = nullptr;
    }
    int sm = 0;
    if (cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sm < 1) sm = 148;
    c->n_sm = sm;
    fold_constants(c);
    *out = c;
    return TBSMA_OK;
}

int tbsma_destroy(tbsma_ctx *c)
{
    if (!c) return TBSMA_EINVAL;
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->graph_exec_multi) cudaGraphExecDestroy(c->graph_exec_multi);
    free_system(c);
    free_staging(c);
    if (c->own_stream) cudaStreamDestroy(c->own_stream);
    if (c->aux_stream) cudaStreamDestroy(c->aux_stream);
    if (c->body_stream) cudaStreamDestroy(c->body_stream);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->tev) {
        for (int i = 0; i < 6 * TBSMA_TIMING_MAX_STEPS; ++i) if (c->tev[i]) cudaEventDestroy(c->tev[i]);
        free(c->tev);
    }
    free(c);
    return TBSMA_OK;
}

int tbsma_set_variant(tbsma_ctx *c, int32_t variant)
{
    if (!c || variant < 0 || variant > 2) return TBSMA_EINVAL;
    c->epoch++;
    c->tiles_rejected = 0;
    c->variant = variant;
    c->cells_built = c->list_built = 0;   // lists must be rebuilt for the new variant
    return TBSMA_OK;
}

int tbsma_get_variant(const tbsma_ctx *c) { return c ? c->active_variant : TBSMA_EINVAL; }

int tbsma_set_tile(tbsma_ctx *c, int32_t layers_per_tile, int32_t threads)
{
    if (!c || layers_per_tile < 1 || layers_per_tile > TBSMA_TILE_MAX_LAYERS || threads < 32 || threads > 512 ||
        (threads & 31))
        return TBSMA_EINVAL;
    c->epoch++;
    c->tiles_rejected = 0;
    c->tile_layers = layers_per_tile;
    c->tile_threads = threads;
    c->cells_built = c->list_built = 0;
    return TBSMA_OK;
}

int tbsma_set_tile_split(tbsma_ctx *c, int32_t ctas_per_tile)
{
    if (!c || ctas_per_tile < 0 || ctas_per_tile > 128) return TBSMA_EINVAL;
    c->epoch++;
    c->tiles_rejected = 0;
    c->tile_split_req = ctas_per_tile;
    c->cells_built = c->list_built = 0;
    return TBSMA_OK;
}

int tbsma_set_tile_box(tbsma_ctx *c, int32_t force)
{
    if (!c) return TBSMA_EINVAL;
    c->epoch++;
    c->tiles_rejected = 0;
    c->tile_force_box = force != 0;
    c->cells_built = c->list_built = 0;
    return TBSMA_OK;
}

int tbsma_set_fused_step(tbsma_ctx *c, int32_t enable)
{
    if (!c) return TBSMA_EINVAL;
    c->epoch++;
    c->fused_step = enable != 0;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph_exec_multi) { cudaGraphExecDestroy(c->graph_exec_multi); c->graph_exec_multi = nullptr; }
    return TBSMA_OK;
}

int tbsma_set_gather(tbsma_ctx *c, int32_t mode)
{
    if (!c || mode < 0 || mode > 4) return TBSMA_EINVAL;
    c->epoch++;
    c->gather_mode = mode != 0;
    c->p_nb_req = mode >= 2 ? mode : 0;
    c->cells_built = c->list_built = 0;
    return TBSMA_OK;
}

int tbsma_set_outer_skin(tbsma_ctx *c, double outer_skin)
{
    if (!c || !(outer_skin >= 0.0) || !(outer_skin <= 16.0)) return TBSMA_EINVAL;
    c->epoch++;
    c->tiles_rejected = 0;
    if (c->d_olist) {
        cudaDeviceSynchronize();
        cudaFree(c->d_tile_first); cudaFree(c->d_work);
        c->d_tile_first = nullptr; c->d_work = nullptr;
        cudaFree(c->d_olist); cudaFree(c->d_nn_o); cudaFree(c->d_pos_outer); cudaFree(c->d_want_outer);
        c->d_olist = nullptr; c->d_nn_o = nullptr; c->d_pos_outer = nullptr; c->d_want_outer = nullptr;
    }
    c->outer_skin = outer_skin;
    fold_constants(c);
    c->cells_built = c->list_built = 0;
    return TBSMA_OK;
}

int tbsma_set_graph(tbsma_ctx *c, int32_t enable)
{
    if (!c) return TBSMA_EINVAL;
    c->epoch++;
    c->use_graph = enable != 0;
    c->use_cond = enable != 1;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph_exec_multi) { cudaGraphExecDestroy(c->graph_exec_multi); c->graph_exec_multi = nullptr; }
    return TBSMA_OK;
}

int tbsma_set_balance(tbsma_ctx *c, int32_t enable, double cell)
{
    if (!c || cell < 0.0) return TBSMA_EINVAL;
    c->epoch++;
    c->balance = enable != 0;
    c->class_h = cell > 0.0 ? cell : c->prm.r0 / sqrt(2.0);
    return TBSMA_OK;
}

int tbsma_set_thermostat(tbsma_ctx *c, int32_t kind, double tau_fs)
{
    if (!c || kind < 0 || kind > 1 || (kind == 1 && !(tau_fs > 0.0))) return TBSMA_EINVAL;
    c->epoch++;
    c->thermostat_kind = kind;
    c->nh_tau = tau_fs;
    if (c->d_nh) CK(cudaMemset(c->d_nh, 0, sizeof(double) * 2 * (size_t)c->R));
    return TBSMA_OK;
}

int tbsma_get_thermostat(tbsma_ctx *c, double *h_xi, double *h_eta)
{
    if (!c || !h_xi || !h_eta) return TBSMA_EINVAL;
    if (!c->d_nh) return TBSMA_ESTATE;
    CK(cudaDeviceSynchronize());
    double *h = (double *)malloc(sizeof(double) * 2 * (size_t)(c->R ? c->R : 1));
    if (!h) return TBSMA_ENOMEM;
    const cudaError_t e = cudaMemcpy(h, c->d_nh, sizeof(double) * 2 * (size_t)c->R, cudaMemcpyDeviceToHost);
    for (int r = 0; r < c->R && e == cudaSuccess; ++r) { h_xi[r] = h[2 * r]; h_eta[r] = h[2 * r + 1]; }
    free(h);
    CK(e);
    return TBSMA_OK;
}

int tbsma_set_thermostat_state(tbsma_ctx *c, const double *h_xi, const double *h_eta)
{
    if (!c || !h_xi || !h_eta) return TBSMA_EINVAL;
    if (!c->d_nh) return TBSMA_ESTATE;
    CK(cudaDeviceSynchronize());
    double *h = (double *)malloc(sizeof(double) * 2 * (size_t)(c->R ? c->R : 1));
    if (!h) return TBSMA_ENOMEM;
    for (int r = 0; r < c->R; ++r) { h[2 * r] = h_xi[r]; h[2 * r + 1] = h_eta[r]; }
    const cudaError_t e = cudaMemcpy(c->d_nh, h, sizeof(double) * 2 * (size_t)c->R, cudaMemcpyHostToDevice);
    free(h);
    CK(e);
    return TBSMA_OK;
}

int tbsma_set_protocol(tbsma_ctx *c, const tbsma_protocol *p)
{
    if (!c || (p && p->stepwise_period < 0)) return TBSMA_EINVAL;
    c->epoch++;
    if (p) c->proto = *p;
    else memset(&c->proto, 0, sizeof(c->proto));
    return TBSMA_OK;
}

int tbsma_set_series(tbsma_ctx *c, const tbsma_series *s)
{
    if (!c) return TBSMA_EINVAL;
    if (s && s->every > 0 && (s->capacity < 1 || !s->d_series || !s->d_count || !s->d_volume || !s->d_L0)) return TBSMA_EINVAL;
    if (s && s->every < 0) return TBSMA_EINVAL;
    c->epoch++;
    if (s && s->every > 0) {
        if (!c->d_geom) return TBSMA_ESTATE;
        if (!c->d_series_w) CK(dalloc(&c->d_series_w, (size_t)6 * c->R));
        c->series = *s;
    } else {
        memset(&c->series, 0, sizeof(c->series));
    }
    return TBSMA_OK;
}

int tbsma_series_histogram(tbsma_ctx *c, const double *d_series, const int32_t *d_count, int32_t capacity, int32_t col_x,
                           int32_t col_y, double x_lo, double x_hi, int32_t nx, double y_lo, double y_hi, int32_t ny,
                           uint64_t *d_hist, void *stream)
{
    if (!c || !d_series || !d_count || !d_hist || capacity < 1 || col_x < 0 || col_x > 3 || col_y < 0 || col_y > 3 ||
        nx < 1 || ny < 1 || !(x_hi > x_lo) || !(y_hi > y_lo))
        return TBSMA_EINVAL;
    if (!c->d_geom) return TBSMA_ESTATE;
    CK(tbsma_launch_series_histogram(c, d_series, d_count, capacity, col_x, col_y, x_lo, x_hi, nx, y_lo, y_hi, ny,
                                     (unsigned long long *)d_hist, (cudaStream_t)stream));
    return TBSMA_OK;
}

int tbsma_set_stagger(tbsma_ctx *c, int32_t enable)
{
    if (!c) return TBSMA_EINVAL;
    c->epoch++;
    c->stagger = enable != 0;
    return TBSMA_OK;
}

int tbsma_set_async(tbsma_ctx *c, int32_t enable, double margin)
{
    if (!c || margin < 0.0) return TBSMA_EINVAL;
    c->epoch++;
    c->async_inner = enable != 0;
    c->async_margin = margin;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph_exec_multi) { cudaGraphExecDestroy(c->graph_exec_multi); c->graph_exec_multi = nullptr; }
    return TBSMA_OK;
}

int tbsma_set_overlap(tbsma_ctx *c, int32_t enable)
{
    if (!c) return TBSMA_EINVAL;
    c->epoch++;
    c->overlap = enable;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph_exec_multi) { cudaGraphExecDestroy(c->graph_exec_multi); c->graph_exec_multi = nullptr; }
    return TBSMA_OK;
}

int tbsma_set_timing(tbsma_ctx *c, int32_t enable)
{
    if (!c) return TBSMA_EINVAL;
    c->epoch++;
    if (enable && !c->tev) {
        c->tev = (cudaEvent_t *)calloc(6 * TBSMA_TIMING_MAX_STEPS, sizeof(cudaEvent_t));
        if (!c->tev) return TBSMA_ENOMEM;
        for (int i = 0; i < 6 * TBSMA_TIMING_MAX_STEPS; ++i) CK(cudaEventCreate(&c->tev[i]));
    }
    c->timing = enable != 0;
    c->tev_steps = 0;
    return TBSMA_OK;
}

int tbsma_get_timing(tbsma_ctx *c, double *h_ms_sum5, int64_t *h_steps)
{
    if (!c || !h_ms_sum5 || !h_steps) return TBSMA_EINVAL;
    for (int k = 0; k < 5; ++k) h_ms_sum5[k] = 0.0;
    *h_steps = 0;
    if (!c->tev || c->tev_steps == 0) return TBSMA_OK;
    CK(cudaEventSynchronize(c->tev[6 * (c->tev_steps - 1) + 5]));
    for (int s = 0; s < c->tev_steps; ++s)
        for (int k = 0; k < 5; ++k) {
            float ms = 0.f;
            CK(cudaEventElapsedTime(&ms, c->tev[6 * s + k], c->tev[6 * s + k + 1]));
            h_ms_sum5[k] += (double)ms;
        }
    *h_steps = c->tev_steps;
    c->tev_steps = 0;
    return TBSMA_OK;
}

int64_t tbsma_launch_count(const tbsma_ctx *c) { return c ? c->launches : 0; }

int tbsma_set_system(tbsma_ctx *c, int64_t n_atoms, int32_t n_replicas, const int32_t *h_off,
                     const float *h_lo, const float *h_hi, const uint8_t *h_per, int32_t max_neighbors)
{
    if (!c || n_atoms < 0 || n_atoms > 0x7ffffff0ll || n_replicas < 1 || !h_off || !h_lo || !h_hi || !h_per ||
        max_neighbors < 1 || max_neighbors > 4096)
        return TBSMA_EINVAL;
    c->epoch++;
    c->tiles_rejected = 0;
    if (h_off[0] != 0 || h_off[n_replicas] != n_atoms) return TBSMA_EINVAL;
    for (int r = 0; r < n_replicas; ++r)
        if (h_off[r + 1] < h_off[r]) return TBSMA_EINVAL;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph_exec_multi) { cudaGraphExecDestroy(c->graph_exec_multi); c->graph_exec_multi = nullptr; }
    free_system(c);
    const int R = n_replicas;
    c->n = n_atoms;
    c->R = R;
    c->n_pad = (int)((n_atoms + 31) / 32 * 32);
    if (c->n_pad < 32) c->n_pad = 32;
    c->kmax = (max_neighbors + 3) / 4 * 4;
    c->launches = 0;
    c->h_off = (int32_t *)malloc(sizeof(int32_t) * (R + 1));
    c->h_geom = (RepGeom *)calloc(R, sizeof(RepGeom));
    if (!c->h_off || !c->h_geom) { free_system(c); return TBSMA_ENOMEM; }
    memcpy(c->h_off, h_off, sizeof(int32_t) * (R + 1));
    const double r_list = c->r_cut + c->skin;
    c->any_periodic = 0;
    for (int r = 0; r < R; ++r) {
        RepGeom &g = c->h_geom[r];
        g.periodic = 0;
        for (int a = 0; a < 3; ++a) {
            const float lo = h_lo[3 * r + a], hi = h_hi[3 * r + a];
            const float len = hi - lo;          // fp32 difference
            if (!(len >= 0.0f) || !isfinite(len)) { free_system(c); return TBSMA_EINVAL; }
            if (h_per[3 * r + a] != 0) {
                if ((double)len < 2.0 * r_list) { free_system(c); return TBSMA_EINVAL; }
                g.periodic |= 1 << a;
                c->any_periodic = 1;
            }
            g.lo[a] = lo;
            g.len[a] = len;
        }
        g.atom_begin = h_off[r];
        g.atom_end = h_off[r + 1];
    }
    const size_t n = (size_t)n_atoms;
    cudaError_t e = cudaSuccess;
#define DA(ptr, cnt) if (e == cudaSuccess) e = dalloc(&(ptr), (cnt))
    DA(c->d_geom, (size_t)R); DA(c->d_atom_rep, n); DA(c->d_cell_of, n); DA(c->d_slot, n); DA(c->d_order, n);
    c->list_bufs = 2;   // the tile variant double-buffers its lists (the global variant uses the first half)
    const size_t nb = (size_t)c->list_bufs;
    DA(c->d_pos_build, nb * c->n_pad); DA(c->d_tmp4, n); DA(c->d_tmp_tag, n);
    DA(c->d_nlist, nb * (size_t)c->kmax * (size_t)c->n_pad); DA(c->d_nn, nb * c->n_pad); DA(c->d_xs, n);
    int64_t n_blk = 0;
    for (int r = 0; r < R; ++r) n_blk += (h_off[r + 1] - h_off[r] + 255) / 256;
    c->n_blk = (int)n_blk;
    DA(c->d_cur, (size_t)R); DA(c->d_nh, 2 * (size_t)R); DA(c->d_kmid, 2 * (size_t)n_blk); DA(c->d_nh_scale, (size_t)R);
    DA(c->d_blk_rep, (size_t)n_blk); DA(c->d_blk_first, (size_t)R + 1);
    DA(c->d_dirty, (size_t)R); DA(c->d_ctrl, 8); DA(c->d_counters, 8); DA(c->d_stagger, (size_t)R);
    DA(c->d_maxpop, 2 * (size_t)R); DA(c->d_hbase, n); DA(c->d_tileof, n); DA(c->d_newslot, n); DA(c->d_oldof, n); DA(c->d_nn_tmp, n);
    DA(c->d_tmp_pos, n);
#undef DA
    if (e != cudaSuccess) { free_system(c); return map_cuda(e); }
    int32_t *rep = (int32_t *)malloc(sizeof(int32_t) * (n ? n : 1));
    if (!rep) { free_system(c); return TBSMA_ENOMEM; }
    for (int r = 0; r < R; ++r)
        for (int64_t i = h_off[r]; i < h_off[r + 1]; ++i) rep[i] = r;
    e = cudaMemcpy(c->d_atom_rep, rep, sizeof(int32_t) * n, cudaMemcpyHostToDevice);
    free(rep);
    {   // runs of 256 consecutive atoms of one replica (ordered sums of the Nose-Hoover kinetic energy)
        int32_t *br = (int32_t *)malloc(sizeof(int32_t) * (size_t)(n_blk ? n_blk : 1));
        int32_t *bf = (int32_t *)malloc(sizeof(int32_t) * (size_t)(R + 1));
        if (!br || !bf) { free(br); free(bf); free_system(c); return TBSMA_ENOMEM; }
        int64_t k = 0;
        for (int r = 0; r < R; ++r) {
            bf[r] = (int32_t)k;
            for (int64_t b = 0; b < (h_off[r + 1] - h_off[r] + 255) / 256; ++b) br[k++] = r;
        }
        bf[R] = (int32_t)k;
        if (e == cudaSuccess) e = cudaMemcpy(c->d_blk_rep, br, sizeof(int32_t) * (size_t)n_blk, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(c->d_blk_first, bf, sizeof(int32_t) * (size_t)(R + 1), cudaMemcpyHostToDevice);
        free(br); free(bf);
    }
    if (e == cudaSuccess) e = cudaMemset(c->d_dirty, 0, sizeof(int32_t) * R);
    if (e == cudaSuccess) e = cudaMemset(c->d_stagger, 0, sizeof(float) * R);
    if (e == cudaSuccess) e = cudaMemset(c->d_ctrl, 0, sizeof(int32_t) * 8);
    if (e == cudaSuccess) e = cudaMemset(c->d_counters, 0, sizeof(unsigned long long) * 8);
    if (e == cudaSuccess) e = cudaMemset(c->d_nn, 0, sizeof(int32_t) * nb * (c->n_pad ? c->n_pad : 1));
    if (e == cudaSuccess) e = cudaMemset(c->d_cur, 0, sizeof(int32_t) * R);
    if (e == cudaSuccess) e = cudaMemset(c->d_nh, 0, sizeof(double) * 2 * R);
    if (e != cudaSuccess) { free_system(c); return map_cuda(e); }
    c->cell_w = 0.0;
    c->kmax_o = c->kmax;
    const int rc = set_geometry(c, tiles_possible(c) ? r_list + c->outer_skin : r_list);
    if (rc) { free_system(c); return rc; }
    return TBSMA_OK;
}

int tbsma_build_cells(tbsma_ctx *c, float *d_pos, float *d_vel, int32_t *d_tag, void *stream)
{
    if (!c || !d_pos || !d_tag) return TBSMA_EINVAL;
    c->epoch++;
    if (!c->d_geom) return TBSMA_ESTATE;
    if (c->n == 0) { c->cells_built = 1; return TBSMA_OK; }
    cudaStream_t st = (cudaStream_t)stream;
    c->list_built = 0;
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
    if (c->graph_exec_multi) { cudaGraphExecDestroy(c->graph_exec_multi); c->graph_exec_multi = nullptr; }   // tiles may change
    {
        const int rc0 = ensure_variant_resources(c);
        if (rc0) return rc0;
    }
    c->active_variant = tiles_possible(c) ? 2 : 1;   // provisional: selects the dirty level
    // every list is rebuilt from here on: all replicas start from half 0 of the list buffers again (the global variant
    // only ever uses half 0; after a run in the tile variant some replicas would otherwise still point at half 1)
    CK(cudaMemsetAsync(c->d_cur, 0, sizeof(int32_t) * (size_t)c->R, st));
    CK(tbsma_launch_mark_all_dirty(c, st));
    CK(tbsma_launch_rebuild(c, (float4 *)d_pos, (float4 *)d_vel, d_tag, true, false, st));
    const int rc = tbsma_tile_setup(c, st);   // picks the gather variant for these cells (synchronises)
    if (rc) return rc;
    if (c->active_variant == 1 && c->cell_w != c->r_cut + c->skin) {
        // the tiles were tried and not taken: the global variant wants its own, narrower cells (fewer candidates per atom
        // in its list build), so bin once more
        c->tiles_rejected = 1;      // (remembered until the system or a tile setting changes: later builds bin once)
        CK(cudaStreamSynchronize(st));
        const int rg = set_geometry(c, c->r_cut + c->skin);
        if (rg) return rg;
        CK(tbsma_launch_mark_all_dirty(c, st));
        CK(tbsma_launch_rebuild(c, (float4 *)d_pos, (float4 *)d_vel, d_tag, true, false, st));
    }
    c->cells_built = 1;
    return TBSMA_OK;
}

int tbsma_build_neighbors(tbsma_ctx *c, float *d_pos, float *d_vel, int32_t *d_tag, void *stream)
{
    if (!c || !d_pos || !d_tag) return TBSMA_EINVAL;
    c->epoch++;
    if (!c->d_geom || !c->cells_built) return TBSMA_ESTATE;
    if (c->n == 0) { c->list_built = 1; return TBSMA_OK; }
    cudaStream_t st = (cudaStream_t)stream;
    CK(tbsma_launch_mark_all_dirty(c, st));
    if (c->active_variant == 2) CK(tbsma_launch_tile_worklist(c, st));
    CK(tbsma_launch_rebuild(c, (float4 *)d_pos, (float4 *)d_vel, d_tag, false, true, st));
    if (c->active_variant == 2) CK(tbsma_launch_tile_inner(c, (const float4 *)d_pos, 1, st));
    CK(tbsma_launch_finish_step(c, 0, st));
    CK(tbsma_launch_set_stagger(c, st));
    c->list_built = 1;
    return TBSMA_OK;
}

int tbsma_compute(tbsma_ctx *c, const float *d_pos, float *d_force_energy, double *d_e, double *d_w, void *stream)
{
    if (!c || !d_pos || !d_force_energy) return TBSMA_EINVAL;
    if (!c->d_geom || !c->list_built) return TBSMA_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    if (d_e) CK(cudaMemsetAsync(d_e, 0, sizeof(double) * c->R, st));
    if (d_w) CK(cudaMemsetAsync(d_w, 0, sizeof(double) * 6 * c->R, st));
    if (c->n == 0) return TBSMA_OK;
    KickArgs kk = {nullptr, 0.f, 0.f, nullptr};
    if (c->active_variant == 2) {
        CK(tbsma_launch_density_tile(c, (const float4 *)d_pos, 1, st));
        CK(tbsma_launch_force_tile(c, (float4 *)d_force_energy, d_w != nullptr, kk, 1, st));
        CK(tbsma_launch_reduce_replicas(c, d_e, nullptr, d_w, st));
    } else {
        CK(tbsma_launch_density(c, (const float4 *)d_pos, st));
        CK(tbsma_launch_force(c, (float4 *)d_force_energy, d_e, d_w, kk, st));
    }
    return TBSMA_OK;
}

int tbsma_md_step(tbsma_ctx *c, float *d_pos, float *d_vel, float *d_force_energy, int32_t *d_tag, double dt_fs,
                  const float *d_T, double gamma_per_fs, const uint64_t *d_seed, uint64_t step,
                  const double *d_slab_disp, double *d_e, double *d_w, double *d_k, void *stream)
{
    if (!c || !d_pos || !d_vel || !d_force_energy || !d_tag || !(dt_fs > 0.0) || !(gamma_per_fs >= 0.0)) return TBSMA_EINVAL;
    if (c && c->thermostat_kind == 0 && gamma_per_fs > 0.0 && (!d_T || !d_seed)) return TBSMA_EINVAL;
    if (c && c->thermostat_kind == 1 && !d_T) return TBSMA_EINVAL;
    if (!c->d_geom || !c->list_built) return TBSMA_ESTATE;
    if (c->n == 0) return TBSMA_OK;
    return run_steps(c, (float4 *)d_pos, (float4 *)d_vel, (float4 *)d_force_energy, d_tag, dt_fs, d_T, gamma_per_fs,
                     (const unsigned long long *)d_seed, step, 1, d_slab_disp, nullptr, 0, d_e, d_w, d_k, false,
                     (cudaStream_t)stream);
}

int tbsma_md_run(tbsma_ctx *c, float *d_pos, float *d_vel, float *d_force_energy, int32_t *d_tag, double dt_fs,
                 const float *d_T, double gamma_per_fs, const uint64_t *d_seed, uint64_t step0, int64_t n_steps,
                 const double *d_disp0, const double *d_rate, int32_t rebuild_every, double *d_e, double *d_w,
                 double *d_k, void *stream)
{
    if (!c || !d_pos || !d_vel || !d_force_energy || !d_tag || !(dt_fs > 0.0) || !(gamma_per_fs >= 0.0) ||
        n_steps < 0 || rebuild_every < 0)
        return TBSMA_EINVAL;
    if (c && c->thermostat_kind == 0 && gamma_per_fs > 0.0 && (!d_T || !d_seed)) return TBSMA_EINVAL;
    if (c && c->thermostat_kind == 1 && !d_T) return TBSMA_EINVAL;
    if (!c->d_geom || !c->list_built) return TBSMA_ESTATE;
    if (c->n == 0 || n_steps == 0) return TBSMA_OK;
    cudaStream_t st = (cudaStream_t)stream;
    float4 *pos = (float4 *)d_pos, *vel = (float4 *)d_vel, *force = (float4 *)d_force_energy;
    const unsigned long long *seed = (const unsigned long long *)d_seed;
    CK(cudaMemsetAsync(c->d_counters, 0, sizeof(unsigned long long), st));   // in-run step offset = 0
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (st) cudaStreamIsCapturing(st, &cap);
    const bool graph = c->use_graph && !c->timing && st != nullptr && cap == cudaStreamCaptureStatusNone && n_steps >= 8;
    if (!graph) {
        int rc = run_steps(c, pos, vel, force, d_tag, dt_fs, d_T, gamma_per_fs, seed, step0, n_steps, d_disp0, d_rate,
                           rebuild_every, d_e, d_w, d_k, true, st);
        if (rc) return rc;
    } else {
        // One step captured into a CUDA graph and replayed: the step counter lives on the device
        // (d_counters[0]), so every replay integrates the next step.  Cached while the arguments repeat.
        GraphKey key;
        memset(&key, 0, sizeof(key));
        key.p[0] = pos; key.p[1] = vel; key.p[2] = force; key.p[3] = d_tag; key.p[4] = d_T; key.p[5] = seed;
        key.p[6] = d_disp0; key.p[7] = d_rate; key.p[8] = d_e; key.p[9] = d_w; key.p[10] = d_k;
        key.dt = dt_fs; key.gamma = gamma_per_fs; key.rebuild_every = rebuild_every;
        key.epoch = c->epoch;
        if (!c->graph_exec || memcmp(&key, &c->graph_key, sizeof(key)) != 0) {
            if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
            if (c->graph_exec_multi) { cudaGraphExecDestroy(c->graph_exec_multi); c->graph_exec_multi = nullptr; }
            // A small batch (the fused step, a few tens of microseconds) pays as much for the launch of a graph as for a
            // kernel: eight steps are captured into a second graph, replayed n / 8 times; the one-step graph takes the rest.
            const int multi = c->active_variant == 2 && tbsma_step_small_ok(c) ? 8 : 1;
            for (int which = 0; which < (multi > 1 ? 2 : 1); ++which) {
                cudaGraph_t g = nullptr;
                CK(cudaStreamBeginCapture(st, cudaStreamCaptureModeThreadLocal));
                const int64_t before = c->launches;
                int rc = run_steps(c, pos, vel, force, d_tag, dt_fs, d_T, gamma_per_fs, seed, 0, which ? multi : 1, d_disp0,
                                   d_rate, rebuild_every, d_e, d_w, d_k, true, st, true);
                cudaError_t e = cudaStreamEndCapture(st, &g);
                if (!which) c->graph_launches_per_step = c->launches - before;
                c->launches = before;
                if (rc) { if (g) cudaGraphDestroy(g); return rc; }
                if (e != cudaSuccess) return map_cuda(e);
                e = cudaGraphInstantiate(which ? &c->graph_exec_multi : &c->graph_exec, g, 0);
                cudaGraphDestroy(g);
                if (e != cudaSuccess) {
                    if (which) c->graph_exec_multi = nullptr; else c->graph_exec = nullptr;
                    return map_cuda(e);
                }
            }
            c->graph_multi_steps = multi;
            c->graph_key = key;
        }
        // the captured step reads the number of the run's first step from the device: one graph serves every step0
        CK(tbsma_launch_set_step_base(c, step0, st));
        int64_t s = 0;
        if (c->graph_exec_multi)
            for (; s + c->graph_multi_steps <= n_steps; s += c->graph_multi_steps) CK(cudaGraphLaunch(c->graph_exec_multi, st));
        for (; s < n_steps; ++s) CK(cudaGraphLaunch(c->graph_exec, st));
        c->launches += c->graph_launches_per_step * n_steps;
    }
    CK(cudaMemsetAsync(c->d_counters, 0, sizeof(unsigned long long), st));
    return TBSMA_OK;
}

int tbsma_md_run_host(tbsma_ctx *c, float *h_pos, float *h_vel, float *h_force, int32_t *h_tag, double dt_fs,
                      const float *h_T, double gamma_per_fs, const uint64_t *h_seed, uint64_t step0, int64_t n_steps,
                      const double *h_disp0, const double *h_rate, int32_t rebuild_every, double *h_e, double *h_w,
                      double *h_k)
{
    if (!c || !h_pos || !h_vel || !h_force || !h_tag || !h_T || !h_seed) return TBSMA_EINVAL;
    if (!c->d_geom) return TBSMA_ESTATE;
    const size_t n = (size_t)c->n;
    const int R = c->R;
    if (!c->own_stream) CK(cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking));
    cudaStream_t st = c->own_stream;
    if (c->s_n != c->n || c->s_R != R) {
        free_staging(c);
        cudaError_t e = cudaSuccess;
#define DA(ptr, cnt) if (e == cudaSuccess) e = dalloc(&(ptr), (cnt))
        DA(c->s_pos, n); DA(c->s_vel, n); DA(c->s_force, n); DA(c->s_tag, n); DA(c->s_T, (size_t)R);
        DA(c->s_seed, (size_t)R); DA(c->s_disp0, (size_t)R); DA(c->s_rate, (size_t)R); DA(c->s_e, (size_t)R);
        DA(c->s_w, (size_t)6 * R); DA(c->s_k, (size_t)R);
#undef DA
        if (e != cudaSuccess) { free_staging(c); return map_cuda(e); }
        c->s_n = c->n; c->s_R = R;
    }
    const cudaMemcpyKind H2D = cudaMemcpyHostToDevice, D2H = cudaMemcpyDeviceToHost;
    CK(cudaMemcpyAsync(c->s_pos, h_pos, 16 * n, H2D, st));
    CK(cudaMemcpyAsync(c->s_vel, h_vel, 16 * n, H2D, st));
    CK(cudaMemcpyAsync(c->s_tag, h_tag, 4 * n, H2D, st));
    CK(cudaMemcpyAsync(c->s_T, h_T, 4 * (size_t)R, H2D, st));
    CK(cudaMemcpyAsync(c->s_seed, h_seed, 8 * (size_t)R, H2D, st));
    if (h_disp0) CK(cudaMemcpyAsync(c->s_disp0, h_disp0, 8 * (size_t)R, H2D, st));
    if (h_rate) CK(cudaMemcpyAsync(c->s_rate, h_rate, 8 * (size_t)R, H2D, st));
    int rc = tbsma_build_cells(c, (float *)c->s_pos, (float *)c->s_vel, c->s_tag, st);
    if (!rc) rc = tbsma_build_neighbors(c, (float *)c->s_pos, (float *)c->s_vel, c->s_tag, st);
    if (!rc) rc = tbsma_compute(c, (float *)c->s_pos, (float *)c->s_force, c->s_e, h_w ? c->s_w : nullptr, st);
    if (!rc) rc = tbsma_md_run(c, (float *)c->s_pos, (float *)c->s_vel, (float *)c->s_force, c->s_tag, dt_fs, c->s_T,
                               gamma_per_fs, (const uint64_t *)c->s_seed, step0, n_steps, h_disp0 ? c->s_disp0 : nullptr,
                               h_rate ? c->s_rate : nullptr, rebuild_every, c->s_e, h_w ? c->s_w : nullptr, c->s_k, st);
    if (rc) return rc;
    CK(cudaMemcpyAsync(h_pos, c->s_pos, 16 * n, D2H, st));
    CK(cudaMemcpyAsync(h_vel, c->s_vel, 16 * n, D2H, st));
    CK(cudaMemcpyAsync(h_force, c->s_force, 16 * n, D2H, st));
    CK(cudaMemcpyAsync(h_tag, c->s_tag, 4 * n, D2H, st));
    if (h_e) CK(cudaMemcpyAsync(h_e, c->s_e, 8 * (size_t)R, D2H, st));
    if (h_w) CK(cudaMemcpyAsync(h_w, c->s_w, 48 * (size_t)R, D2H, st));
    if (h_k) CK(cudaMemcpyAsync(h_k, c->s_k, 8 * (size_t)R, D2H, st));
    CK(cudaStreamSynchronize(st));
    return TBSMA_OK;
}

int tbsma_kinetic_tensor(tbsma_ctx *c, const float *d_pos, const float *d_vel, double *d_k, void *stream)
{
    if (!c || !d_pos || !d_vel || !d_k) return TBSMA_EINVAL;
    if (!c->d_geom) return TBSMA_ESTATE;
    if (c->n == 0) return TBSMA_OK;
    CK(tbsma_launch_kinetic_tensor(c, (const float4 *)d_pos, (const float4 *)d_vel, d_k, (cudaStream_t)stream));
    return TBSMA_OK;
}

int tbsma_stress(tbsma_ctx *c, const double *d_w, const double *d_k, const double *d_volume, double *d_sigma, void *stream)
{
    if (!c || !d_w || !d_volume || !d_sigma) return TBSMA_EINVAL;
    if (!c->d_geom) return TBSMA_ESTATE;
    if (c->R == 0) return TBSMA_OK;
    CK(tbsma_launch_stress(c, d_w, d_k, d_volume, d_sigma, (cudaStream_t)stream));
    return TBSMA_OK;
}

int tbsma_get_neighbors(tbsma_ctx *c, const int32_t *d_tag, int32_t *d_counts, int32_t *d_list, void *stream)
{
    if (!c || !d_tag || !d_counts || !d_list) return TBSMA_EINVAL;
    if (!c->list_built) return TBSMA_ESTATE;
    if (c->n == 0) return TBSMA_OK;
    if (c->active_variant == 2) CK(tbsma_launch_get_neighbors_tile(c, d_tag, d_counts, d_list, (cudaStream_t)stream));
    else CK(tbsma_launch_get_neighbors(c, d_tag, d_counts, d_list, (cudaStream_t)stream));
    return TBSMA_OK;
}

int tbsma_count_pairs(tbsma_ctx *c, const float *d_pos, int64_t *h_entries, int64_t *h_pairs, void *stream)
{
    if (!c || !d_pos) return TBSMA_EINVAL;
    if (!c->list_built) return TBSMA_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned long long out[2] = {0, 0};
    if (c->n > 0) {
        CK(cudaMemsetAsync(c->d_counters + 4, 0, 2 * sizeof(unsigned long long), st));
        if (c->active_variant == 2) CK(tbsma_launch_count_pairs_tile(c, (const float4 *)d_pos, c->d_counters + 4, st));
        else CK(tbsma_launch_count_pairs(c, (const float4 *)d_pos, c->d_counters + 4, st));
        CK(cudaMemcpyAsync(out, c->d_counters + 4, sizeof(out), cudaMemcpyDeviceToHost, st));
        CK(cudaStreamSynchronize(st));
    }
    if (h_entries) *h_entries = (int64_t)out[0];
    if (h_pairs) *h_pairs = (int64_t)out[1];
    return TBSMA_OK;
}

int tbsma_status(tbsma_ctx *c, uint32_t *h_flags)
{
    if (!c || !h_flags) return TBSMA_EINVAL;
    *h_flags = 0;
    if (!c->d_ctrl) return TBSMA_OK;
    CK(cudaDeviceSynchronize());
    int v = 0;
    CK(cudaMemcpy(&v, c->d_ctrl + 1, sizeof(int), cudaMemcpyDeviceToHost));
    *h_flags = (uint32_t)v;
    return TBSMA_OK;
}

int tbsma_clear_status(tbsma_ctx *c)
{
    if (!c) return TBSMA_EINVAL;
    if (!c->d_ctrl) return TBSMA_OK;
    CK(cudaDeviceSynchronize());
    CK(cudaMemset(c->d_ctrl + 1, 0, sizeof(int)));
    return TBSMA_OK;
}

int tbsma_get_stats(tbsma_ctx *c, tbsma_stats *out)
{
    if (!c || !out) return TBSMA_EINVAL;
    memset(out, 0, sizeof(*out));
    if (!c->d_ctrl) return TBSMA_OK;
    CK(cudaDeviceSynchronize());
    unsigned long long cnt[8];
    int ctrl[4];
    CK(cudaMemcpy(cnt, c->d_counters, sizeof(cnt), cudaMemcpyDeviceToHost));
    CK(cudaMemcpy(ctrl, c->d_ctrl, sizeof(ctrl), cudaMemcpyDeviceToHost));
    out->n_steps = cnt[3];
    out->n_replica_builds = cnt[1];
    out->n_build_passes = cnt[2];
    out->max_neighbors_seen = ctrl[2];
    out->n_candidate_builds = (int32_t)(cnt[6] > 0x7fffffffull ? 0x7fffffffull : cnt[6]);
    return TBSMA_OK;
}

}  // extern "C"
