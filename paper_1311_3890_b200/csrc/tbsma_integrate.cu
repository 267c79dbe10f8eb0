// tbsma_integrate.cu -- the first half of the MD step and the step bookkeeping.
//
// "the equations of motion are integrated using the velocity Verlet algorithm with a time
// step of 2.0 fs"; "Two rigid layers of gripping atoms ... are periodically displaced".  The
// paper's thermostat is Nose-Hoover; BASELINE.json substitutes Langevin with a counter-based
// Philox generator, discretised as BAOAB (D:A8), which is exactly velocity Verlet for gamma = 0:
//   B: v += (dt/2)(c/m) F    A: x += (dt/2) v    O: v <- c1 v + c2 sigma_v g    A: x += (dt/2) v
// (forces and the closing B run in tbsma_force.cu).  The same kernel measures every atom's
// displacement since the last list build and raises its replica's dirty flag (D:A14).
#include "tbsma_integrate.cuh"

namespace {

__global__ void __launch_bounds__(256)
k_integrate_pre(float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ force,
                const float4 *__restrict__ pos_build, const int *__restrict__ atom_rep,
                const RepGeom *__restrict__ geom, const int *__restrict__ tag, StepArgs a,
                const unsigned long long *__restrict__ counters, int *__restrict__ dirty,
                int *__restrict__ ctrl, int n, int R)
{
    tbsma_integrate_one(blockIdx.x * blockDim.x + threadIdx.x, pos, vel, force, pos_build, atom_rep, geom, tag, a, counters,
                        dirty, ctrl, n, R);
}

// end of step: statistics, clear the dirty flags, advance the in-run step offset
__global__ void __launch_bounds__(256)
k_finish_step(int *__restrict__ dirty, int *__restrict__ ctrl, int *__restrict__ want_outer,
              float *__restrict__ stagger, int *__restrict__ cur, int swap,
              unsigned long long *__restrict__ counters, int R, int advance, int count_step, TileSums ts)
{
    tbsma_reduce_replicas(ts, R);      // a6 of the tile variant: per-replica E, E_kin, W in a fixed order (all CTAs)
    if (blockIdx.x != 0) return;       // the bookkeeping below is CTA 0's
    tbsma_finish_bookkeeping(dirty, ctrl, stagger, cur, swap, counters, R, advance, count_step);
}

// Replicas that are built together (all of them, at the start of a run) and share a temperature would all ask
// for their next list at nearly the same step, and again one period later: steps with a hundred rebuilds
// between steps with none.  Rebuilding early is always valid, so until its first rebuild replica r uses the
// fraction f_r^2 of (skin/2)^2, f_r = 0.3 + 0.7 frac(r phi): the rebuild phases start out spread evenly.
__global__ void k_set_stagger(float *__restrict__ stagger, int R, int enable)
{
    const int r = blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= R) return;
    float f = 1.0f;
    if (enable && R > 1) {
        const float u = (float)r * 0.6180339887f;
        f = 0.3f + 0.7f * (u - floorf(u));
    }
    stagger[r] = f * f;
}

// ---- Nose-Hoover (the paper's thermostat; reading A17): B A N A B with one variable xi per replica,
//   N:  xi += (dt/2)(2K - g kB T)/Q;  v *= s = exp(-xi dt);  K *= s^2;  xi += (dt/2)(2K - g kB T)/Q;   Q = g kB T tau^2,
// K = kinetic energy of the dynamic atoms AFTER the opening kick, g = 3 N_dyn.  K needs all atoms of the replica, so it
// is summed by a kernel of its own from (v, F) with the kick of k_integrate_pre, operation for operation; a thread per
// replica then advances xi and eta (d eta/dt = xi: the conserved quantity is E + K + Q xi^2/2 + g kB T eta) and leaves
// the scale for the integrator.
// One CTA per run of 256 consecutive atoms of ONE replica (the runs are laid out by tbsma_set_system: blk_first[r] is
// the first run of replica r), a fixed tree inside the CTA, and k_nh_update adds the runs of a replica in order: the
// kinetic energy that drives xi is bitwise repeatable, and with it the whole Nose-Hoover trajectory.
__global__ void __launch_bounds__(256)
k_nh_kinetic(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const float4 *__restrict__ force,
             const int *__restrict__ blk_rep, const int *__restrict__ blk_first, const RepGeom *__restrict__ geom,
             double *__restrict__ kpart, float kick, double half_m_over_c)
{
    __shared__ double red[2][256];
    const int j = blockIdx.x, r = blk_rep[j];
    const int i = geom[r].atom_begin + 256 * (j - blk_first[r]) + (int)threadIdx.x;
    double k = 0.0, cnt = 0.0;
    if (i < geom[r].atom_end && (__float_as_int(pos[i].w) & 3) == 0) {
        const float4 v = vel[i], f = force[i];
        const double vx = __fmaf_rn(kick, f.x, v.x), vy = __fmaf_rn(kick, f.y, v.y), vz = __fmaf_rn(kick, f.z, v.z);
        k = half_m_over_c * (vx * vx + vy * vy + vz * vz);
        cnt = 1.0;
    }
    red[0][threadIdx.x] = k;
    red[1][threadIdx.x] = cnt;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            red[0][threadIdx.x] += red[0][threadIdx.x + o];
            red[1][threadIdx.x] += red[1][threadIdx.x + o];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) { kpart[2 * (size_t)j] = red[0][0]; kpart[2 * (size_t)j + 1] = red[1][0]; }
}

// a warp per replica: K and the number of dynamic atoms from the runs (lane l adds runs l, l + 32, ... in order, then a
// shuffle tree), then lane 0 advances xi and eta
__global__ void __launch_bounds__(256)
k_nh_update(const double *__restrict__ kpart, const int *__restrict__ blk_first, const float *__restrict__ T,
            const float *__restrict__ T_rate, const unsigned long long *__restrict__ counters,
            double *__restrict__ nh, float *__restrict__ scale, double dt, double tau, int R)
{
    const int r = (int)blockIdx.x * 8 + (int)(threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (r >= R) return;
    double K = 0.0, nd = 0.0;
    for (int j = blk_first[r] + lane; j < blk_first[r + 1]; j += 32) { K += kpart[2 * (size_t)j]; nd += kpart[2 * (size_t)j + 1]; }
    for (int o = 16; o > 0; o >>= 1) {
        K += __shfl_xor_sync(0xffffffffu, K, o);
        nd += __shfl_xor_sync(0xffffffffu, nd, o);
    }
    if (lane != 0) return;
    const double g = 3.0 * nd;
    double Tr = (double)T[r];
    if (T_rate) Tr = fmax(Tr + (double)T_rate[r] * (double)counters[0], 0.0);      // temperature ramp
    const double gkt = g * TBSMA_KB * Tr;
    double s = 1.0;
    if (gkt > 0.0 && tau > 0.0) {
        const double Q = gkt * tau * tau;
        double xi = nh[2 * r];
        xi += 0.5 * dt * (2.0 * K - gkt) / Q;
        s = exp(-xi * dt);
        nh[2 * r + 1] += xi * dt;
        xi += 0.5 * dt * (2.0 * K * s * s - gkt) / Q;
        nh[2 * r] = xi;
    }
    scale[r] = (float)s;
}

// ---- observables of the tensile tests (Eq.5 as read in D:A11) -----------------------
// K_ab = sum_i m v_i,a v_i,b over the dynamic atoms of every replica (eV; xx yy zz xy xz yz).  Atoms of a replica are
// contiguous, so nearly every warp belongs to one replica: warp shuffle sums, one fp64 atomic per warp and component.
__global__ void __launch_bounds__(256)
k_kinetic_tensor(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const int *__restrict__ atom_rep,
                 double *__restrict__ k_rep, double m_over_c, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    const int lane = threadIdx.x & 31;
    int r = -1;
    double k[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (i < n) {
        r = atom_rep[i];
        if ((__float_as_int(pos[i].w) & 3) == 0) {
            const float4 v = vel[i];
            const double vx = v.x, vy = v.y, vz = v.z;
            k[0] = m_over_c * vx * vx; k[1] = m_over_c * vy * vy; k[2] = m_over_c * vz * vz;
            k[3] = m_over_c * vx * vy; k[4] = m_over_c * vx * vz; k[5] = m_over_c * vy * vz;
        }
    }
    const int r0 = __shfl_sync(0xffffffffu, r, 0);
    const bool uniform = __all_sync(0xffffffffu, r == r0);
    if (uniform) {
        if (r0 < 0) return;
#pragma unroll
        for (int c = 0; c < 6; ++c) {
            double s = k[c];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
            if (lane == 0) atomicAdd(k_rep + 6 * (size_t)r0 + c, s);
        }
    } else if (r >= 0) {
#pragma unroll
        for (int c = 0; c < 6; ++c) atomicAdd(k_rep + 6 * (size_t)r + c, k[c]);
    }
}

// sigma_ab = -(W_ab + K_ab) / V, tension positive
__global__ void k_stress(const double *__restrict__ w_rep, const double *__restrict__ k_rep,
                         const double *__restrict__ volume, double *__restrict__ sigma, int R)
{
    const int q = blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= 6 * R) return;
    sigma[q] = -(w_rep[q] + (k_rep ? k_rep[q] : 0.0)) / volume[q / 6];
}

// ---- the tensile test as a device-side series ------------------------------------
// One CTA per replica, after the last kernel of a step of tbsma_md_run.  When a record is due (the number of the step
// just done, plus one, is a multiple of `every`) it appends
//   step | strain (Eq.4: (L - L0) / L0, L - L0 = D_2 - D_1 of the two slabs) | sigma_zz = -(W_zz + K_zz) / V (Eq.5 as read
//   in D:A11, z = the wire axis) | largest gap between consecutive z coordinates of the replica's atoms
// and notes the first step whose gap exceeds r_cut: the wire has parted ("until rupture").  K_zz is added in a fixed
// order (thread-strided partial sums, then a tree).  The gap comes from 2048 bins along z holding the least and the
// greatest z that fell into them: exact whenever it is wider than a bin.  The bins span the z range the replica's atoms
// occupy AT THIS STEP (a first pass finds it), not the box given to tbsma_set_system: a slab pulled beyond the box, and a
// gap that opens out there, are seen like any other.  (A periodic z axis: the gap across the boundary is not looked at.)
#define TBSMA_SERIES_BINS 2048
__device__ __forceinline__ int ord_of(float f) { const int k = __float_as_int(f); return k >= 0 ? k : k ^ 0x7fffffff; }
__device__ __forceinline__ float f_of(int k) { return __int_as_float(k >= 0 ? k : k ^ 0x7fffffff); }

__global__ void __launch_bounds__(256)
k_series_record(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const RepGeom *__restrict__ geom,
                const double *__restrict__ w_rep, const unsigned long long *__restrict__ counters, tbsma_series S,
                StepArgs a, double m_over_c, float r_cut)
{
    __shared__ int s_mn[TBSMA_SERIES_BINS], s_mx[TBSMA_SERIES_BINS];
    __shared__ double s_red[256];
    __shared__ float s_gap[256];
    const unsigned long long nst_done = counters[0];          // steps of this run done, this one included (>= 1)
    const unsigned long long step = (a.step_on_device ? counters[7] : a.step_base) + nst_done - 1ull;
    if ((step + 1ull) % (unsigned long long)S.every != 0ull) return;
    const int r = blockIdx.x, tid = threadIdx.x;
    const int idx = S.d_count[r];
    if (idx >= S.capacity) return;
    const RepGeom *g = geom + r;
    __shared__ int s_zlo, s_zhi;
    for (int b = tid; b < TBSMA_SERIES_BINS; b += 256) { s_mn[b] = 0x7fffffff; s_mx[b] = (int)0x80000000; }
    if (tid == 0) { s_zlo = 0x7fffffff; s_zhi = (int)0x80000000; }
    __syncthreads();
    {
        int zlo = 0x7fffffff, zhi = (int)0x80000000;
        for (int i = g->atom_begin + tid; i < g->atom_end; i += 256) {
            const int o = ord_of(pos[i].z);
            zlo = min(zlo, o);
            zhi = max(zhi, o);
        }
        zlo = __reduce_min_sync(0xffffffffu, zlo);
        zhi = __reduce_max_sync(0xffffffffu, zhi);
        if ((tid & 31) == 0) { atomicMin(&s_zlo, zlo); atomicMax(&s_zhi, zhi); }
    }
    __syncthreads();
    const float z0 = f_of(s_zlo), span = g->atom_end > g->atom_begin ? f_of(s_zhi) - z0 : 0.f;
    const float inv_w = span > 0.f ? (float)TBSMA_SERIES_BINS / span : 0.f;
    double k = 0.0;
    for (int i = g->atom_begin + tid; i < g->atom_end; i += 256) {
        const float4 p = pos[i];
        if ((__float_as_int(p.w) & 3) == 0) {
            const double vz = (double)vel[i].z;
            k += m_over_c * vz * vz;
        }
        int b = __float2int_rd((p.z - z0) * inv_w);
        b = min(max(b, 0), TBSMA_SERIES_BINS - 1);
        const int o = ord_of(p.z);
        atomicMin(&s_mn[b], o);
        atomicMax(&s_mx[b], o);
    }
    s_red[tid] = k;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) s_red[tid] += s_red[tid + o];
        __syncthreads();
    }
    // largest gap between a bin's least z and the greatest z of the nearest occupied bin below it
    float gap = 0.f;
    for (int b = tid; b < TBSMA_SERIES_BINS; b += 256) {
        if (s_mn[b] == 0x7fffffff) continue;
        int q = b - 1;
        while (q >= 0 && s_mn[q] == 0x7fffffff) --q;
        if (q >= 0) gap = fmaxf(gap, f_of(s_mn[b]) - f_of(s_mx[q]));
    }
    s_gap[tid] = gap;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (tid < o) s_gap[tid] = fmaxf(s_gap[tid], s_gap[tid + o]);
        __syncthreads();
    }
    if (tid == 0) {
        unsigned long long nst = nst_done;
        if (a.period > 0) nst = nst / (unsigned long long)a.period * (unsigned long long)a.period;
        double D2 = a.disp0 ? a.disp0[r] : 0.0, D1 = a.disp0_1 ? a.disp0_1[r] : 0.0;
        if (a.rate) D2 += a.rate[r] * (double)nst;
        if (a.rate_1) D1 += a.rate_1[r] * (double)nst;
        double *rec = S.d_series + 4 * ((size_t)r * S.capacity + idx);
        rec[0] = (double)step;
        rec[1] = (D2 - D1) / S.d_L0[r];
        rec[2] = -(w_rep[6 * (size_t)r + 2] + s_red[0]) / S.d_volume[r];
        rec[3] = (double)s_gap[0];
        S.d_count[r] = idx + 1;
        if (S.d_rupture_step && S.d_rupture_step[r] < 0 && s_gap[0] > r_cut) S.d_rupture_step[r] = (long long)step;
    }
}

// stress-strain "heat map" over the records of all replicas (Fig.4): counts per cell of an nx x ny grid over
// [x_lo, x_hi) x [y_lo, y_hi); records outside are not counted
__global__ void k_series_histogram(const double *__restrict__ series, const int *__restrict__ count, int capacity, int R,
                                   int col_x, int col_y, double x_lo, double x_hi, int nx, double y_lo, double y_hi, int ny,
                                   unsigned long long *__restrict__ hist)
{
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= (long long)R * capacity) return;
    const int r = (int)(q / capacity), k = (int)(q % capacity);
    if (k >= count[r]) return;
    const double x = series[4 * q + col_x], y = series[4 * q + col_y];
    if (!(x >= x_lo && x < x_hi && y >= y_lo && y < y_hi)) return;
    int ix = (int)floor((x - x_lo) / (x_hi - x_lo) * (double)nx), iy = (int)floor((y - y_lo) / (y_hi - y_lo) * (double)ny);
    ix = min(ix, nx - 1); iy = min(iy, ny - 1);
    atomicAdd(hist + (size_t)iy * nx + ix, 1ull);
}

}  // namespace

cudaError_t tbsma_launch_series_record(tbsma_ctx *c, const float4 *pos, const float4 *vel, const double *w_rep,
                                       const StepArgs &a, cudaStream_t st)
{
    k_series_record<<<c->R, 256, 0, st>>>(pos, vel, c->d_geom, w_rep, c->d_counters, c->series, a,
                                          c->prm.mass_amu / TBSMA_ACC, (float)c->r_cut);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_series_histogram(tbsma_ctx *c, const double *series, const int32_t *count, int capacity, int col_x,
                                          int col_y, double x_lo, double x_hi, int nx, double y_lo, double y_hi, int ny,
                                          unsigned long long *hist, cudaStream_t st)
{
    const long long total = (long long)c->R * capacity;
    if (total <= 0) return cudaSuccess;
    k_series_histogram<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(series, count, capacity, c->R, col_x, col_y, x_lo, x_hi,
                                                                        nx, y_lo, y_hi, ny, hist);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_nose_hoover(tbsma_ctx *c, const float4 *pos, const float4 *vel, const float4 *force,
                                     const StepArgs &a, double dt, cudaStream_t st)
{
    if (c->n_blk == 0) return cudaSuccess;
    k_nh_kinetic<<<c->n_blk, 256, 0, st>>>(pos, vel, force, c->d_blk_rep, c->d_blk_first, c->d_geom, c->d_kmid, a.kick,
                                           0.5 * c->prm.mass_amu / TBSMA_ACC);
    k_nh_update<<<(c->R + 7) / 8, 256, 0, st>>>(c->d_kmid, c->d_blk_first, a.T, a.T_rate, c->d_counters, c->d_nh,
                                                c->d_nh_scale, dt, c->nh_tau, c->R);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_kinetic_tensor(tbsma_ctx *c, const float4 *pos, const float4 *vel, double *k_rep, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(k_rep, 0, sizeof(double) * 6 * (size_t)c->R, st);
    if (e != cudaSuccess) return e;
    const int n = (int)c->n;
    k_kinetic_tensor<<<(n + 255) / 256, 256, 0, st>>>(pos, vel, c->d_atom_rep, k_rep, c->prm.mass_amu / TBSMA_ACC, n);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_stress(tbsma_ctx *c, const double *w_rep, const double *k_rep, const double *volume,
                                double *sigma, cudaStream_t st)
{
    k_stress<<<(6 * c->R + 255) / 256, 256, 0, st>>>(w_rep, k_rep, volume, sigma, c->R);
    c->launches++;
    return cudaGetLastError();
}

__global__ void k_set_u64(unsigned long long *p, unsigned long long v) { *p = v; }

cudaError_t tbsma_launch_set_step_base(tbsma_ctx *c, unsigned long long step0, cudaStream_t st)
{
    k_set_u64<<<1, 1, 0, st>>>(c->d_counters + 7, step0);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_set_stagger(tbsma_ctx *c, cudaStream_t st)
{
    k_set_stagger<<<(c->R + 255) / 256, 256, 0, st>>>(c->d_stagger, c->R, c->stagger);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_integrate_pre(tbsma_ctx *c, float4 *pos, float4 *vel, const float4 *force,
                                       const int32_t *tag, const StepArgs &a, cudaStream_t st)
{
    const int n = (int)c->n;
    const int work = n > c->R ? n : c->R;
    k_integrate_pre<<<(work + 255) / 256, 256, 0, st>>>(pos, vel, force, c->d_pos_build, c->d_atom_rep, c->d_geom,
                                                        tag, a, c->d_counters, c->d_dirty, c->d_ctrl, n, c->R);
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_finish_step(tbsma_ctx *c, int advance_offset, cudaStream_t st, TileSums ts)
{
    k_finish_step<<<ts.cta_sums ? tbsma_reduce_grid(c->R) : 1, 256, 0, st>>>(c->d_dirty, c->d_ctrl, c->active_variant == 2 ? c->d_want_outer : nullptr,
                                     c->d_stagger, c->d_cur, c->list_bufs == 2 && c->active_variant == 2, c->d_counters, c->R, advance_offset & 1,
                                     (advance_offset >> 1) & 1, ts);
    c->launches++;
    return cudaGetLastError();
}
