// tbsma_force.cu -- the two neighbour-gather passes of the TB-SMA force.
//
// "the total force acting on each atom is calculated in two stages (i.e., two CUDA kernels),
// with each stage looping over atom i's neighbors"; all rho must be complete before stage 2.
//   stage 1 (k_density):  rho_i = sum_j xi^2 exp(-2q(r_ij/r0-1))  (Eq.1); stores
//                         s_i = rho_i^(-1/2) once per atom, packed with the position: (x,y,z,s).
//   stage 2 (k_force):    E_i = sum_j A exp(-p x_ij) - sqrt(rho_i)                (Eq.1-3)
//                         F_i = sum_j [ (2Ap/r0) e^{-p x} - (q xi^2/r0) e^{-2q x} (s_i+s_j) ] d_ij/r_ij
//                         W_ab = 1/2 sum_j d_a f_b   (Eq.5 potential part, D:A11)
// Variant 1 (this file): one thread per atom; the index list is k-major in groups of four
// (int4 per thread per load, 512 B per warp, streamed with ld.global.cs so it does not evict the
// positions); neighbour records are 16-byte gathers served by L1/L2.  Pair math is fp32 with
// MUFU rsqrt/ex2 and constants folded on the host; per-replica sums are fp64.
#include "tbsma_internal.cuh"

namespace {

constexpr int kBlock = 128;

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

struct Box3 { float Lx, Ly, Lz; int per; };

template <bool PERIODIC>
__device__ __forceinline__ void min_image(float &dx, float &dy, float &dz, const Box3 &b)
{
    if (PERIODIC) {
        if (b.per & 1) { const float h = 0.5f * b.Lx; if (dx > h) dx -= b.Lx; else if (dx < -h) dx += b.Lx; }
        if (b.per & 2) { const float h = 0.5f * b.Ly; if (dy > h) dy -= b.Ly; else if (dy < -h) dy += b.Ly; }
        if (b.per & 4) { const float h = 0.5f * b.Lz; if (dz > h) dz -= b.Lz; else if (dz < -h) dz += b.Lz; }
    }
}

// one neighbour of stage 1
template <bool PERIODIC>
__device__ __forceinline__ float rho_term(const float4 &pi, const float4 &pj, bool notself, const Box3 &b,
                                          const PairConst &pc)
{
    float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
    min_image<PERIODIC>(dx, dy, dz, b);
    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));   // D:A6 order
    const bool in = (d2 < pc.rc2) && notself;
    const float rinv = rsqrt_approx(d2);
    const float t = __fmaf_rn(d2, rinv, -pc.r0f);            // r - r0
    const float e = ex2_approx(__fmaf_rn(pc.aq, t, pc.b_rho));
    return in ? e : 0.f;
}

template <bool PERIODIC>
__global__ void __launch_bounds__(kBlock)
k_density(const float4 *__restrict__ pos, const int4 *__restrict__ nlist4, const int *__restrict__ nn,
          const int *__restrict__ atom_rep, const RepGeom *__restrict__ geom, float4 *__restrict__ xs,
          int n, int n_pad /* rows of capacity per atom, kmax / 4 */, PairConst pc)
{
    const int i = blockIdx.x * kBlock + threadIdx.x;
    if (i >= n) return;
    const float4 pi = pos[i];
    const int cnt = nn[i] & 0xffff;
    Box3 b = {0.f, 0.f, 0.f, 0};
    if (PERIODIC) {
        const RepGeom *g = geom + atom_rep[i];
        b.Lx = g->len[0]; b.Ly = g->len[1]; b.Lz = g->len[2]; b.per = g->periodic;
    }
    const int ng = (cnt + 3) >> 2;
    const int4 *row = nlist4 + tbsma_lrow(i, n_pad);
    float rho0 = 0.f, rho1 = 0.f;
    for (int g = 0; g < ng; ++g) {
        const int4 jj = __ldcs(row + (size_t)g * TBSMA_LROW);
        const float4 p0 = pos[jj.x], p1 = pos[jj.y], p2 = pos[jj.z], p3 = pos[jj.w];
        rho0 += rho_term<PERIODIC>(pi, p0, jj.x != i, b, pc);
        rho1 += rho_term<PERIODIC>(pi, p1, jj.y != i, b, pc);
        rho0 += rho_term<PERIODIC>(pi, p2, jj.z != i, b, pc);
        rho1 += rho_term<PERIODIC>(pi, p3, jj.w != i, b, pc);
    }
    const float rho = rho0 + rho1;
    const float s = rho > 0.f ? 1.0f / sqrtf(rho) : 0.f;      // once per atom, IEEE (D:A5 for rho = 0)
    xs[i] = make_float4(pi.x, pi.y, pi.z, s);
}

struct Acc {
    float fx, fy, fz, er;
    float wxx, wyy, wzz, wxy, wxz, wyz;
};

template <bool PERIODIC, bool VIRIAL>
__device__ __forceinline__ void force_term(const float4 &pi, const float4 &pj, bool notself, const Box3 &b,
                                           const PairConst &pc, Acc &a)
{
    float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
    min_image<PERIODIC>(dx, dy, dz, b);
    const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
    const bool in = (d2 < pc.rc2) && notself;
    const float rinv = rsqrt_approx(d2);
    const float t = __fmaf_rn(d2, rinv, -pc.r0f);
    float er = ex2_approx(__fmaf_rn(pc.ap, t, pc.b_rep));        // (2Ap/r0) e^{-p x}
    const float eb = ex2_approx(__fmaf_rn(pc.aq, t, pc.b_band)); // (q xi^2/r0) e^{-2q x}
    float fp = (er - eb * (pi.w + pj.w)) * rinv;                 // -dE/dr / r
    fp = in ? fp : 0.f;
    er = in ? er : 0.f;
    a.fx = __fmaf_rn(fp, dx, a.fx); a.fy = __fmaf_rn(fp, dy, a.fy); a.fz = __fmaf_rn(fp, dz, a.fz);
    a.er += er;
    if (VIRIAL) {
        const float fx = __fmul_rn(fp, dx), fy = __fmul_rn(fp, dy), fz = __fmul_rn(fp, dz);
        a.wxx = __fmaf_rn(dx, fx, a.wxx); a.wyy = __fmaf_rn(dy, fy, a.wyy); a.wzz = __fmaf_rn(dz, fz, a.wzz);
        a.wxy = __fmaf_rn(dx, fy, a.wxy); a.wxz = __fmaf_rn(dx, fz, a.wxz); a.wyz = __fmaf_rn(dy, fz, a.wyz);
    }
}

__device__ __forceinline__ double warp_sum(double v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// a6: add a per-atom value into its replica's fp64 accumulator; one atomic per warp when the
// whole warp belongs to one replica (the common case), per lane at replica boundaries.
__device__ __forceinline__ void replica_add(double *acc, int stride, int comp, int r, bool uniform,
                                            bool active, double v, int lane)
{
    if (uniform) {
        v = warp_sum(active ? v : 0.0);
        if (lane == 0) atomicAdd(acc + (size_t)r * stride + comp, v);
    } else if (active) {
        atomicAdd(acc + (size_t)r * stride + comp, v);
    }
}

template <bool PERIODIC, bool VIRIAL, bool KICK>
__global__ void __launch_bounds__(kBlock)
k_force(const float4 *__restrict__ xs, const int4 *__restrict__ nlist4, const int *__restrict__ nn,
        const int *__restrict__ atom_rep, const RepGeom *__restrict__ geom, float4 *__restrict__ force,
        double *__restrict__ e_rep, double *__restrict__ w_rep, KickArgs kk, int *__restrict__ ctrl,
        int n, int n_pad /* rows of capacity per atom, kmax / 4 */, PairConst pc)
{
    const int i0 = blockIdx.x * kBlock + threadIdx.x;
    const bool active = i0 < n;
    const int i = active ? i0 : n - 1;
    const int lane = threadIdx.x & 31;
    const float4 pi = xs[i];
    const int nni = nn[i];
    const int cnt = active ? (nni & 0xffff) : 0;
    const int r = atom_rep[i];
    Box3 b = {0.f, 0.f, 0.f, 0};
    if (PERIODIC) {
        const RepGeom *g = geom + r;
        b.Lx = g->len[0]; b.Ly = g->len[1]; b.Lz = g->len[2]; b.per = g->periodic;
    }
    const int ng = (cnt + 3) >> 2;
    const int4 *row = nlist4 + tbsma_lrow(i, n_pad);
    Acc a = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
    for (int g = 0; g < ng; ++g) {
        const int4 jj = __ldcs(row + (size_t)g * TBSMA_LROW);
        const float4 p0 = xs[jj.x], p1 = xs[jj.y], p2 = xs[jj.z], p3 = xs[jj.w];
        force_term<PERIODIC, VIRIAL>(pi, p0, jj.x != i, b, pc, a);
        force_term<PERIODIC, VIRIAL>(pi, p1, jj.y != i, b, pc, a);
        force_term<PERIODIC, VIRIAL>(pi, p2, jj.z != i, b, pc, a);
        force_term<PERIODIC, VIRIAL>(pi, p3, jj.w != i, b, pc, a);
    }
    const float sqrt_rho = pi.w > 0.f ? 1.0f / pi.w : 0.f;
    const float ei = __fmaf_rn(a.er, pc.e_rep_scale, -sqrt_rho);   // Eq.1-3: E_R^i + E_B^i
    if (active) {
        force[i] = make_float4(a.fx, a.fy, a.fz, ei);
        if (!isfinite(a.fx + a.fy + a.fz + ei)) atomicOr(ctrl + 1, (int)TBSMA_FLAG_NONFINITE);
    }
    float ke = 0.f;
    if (KICK && active && (nni >> 16) == 0) {     // final B of the step, dynamic atoms only
        float4 v = kk.vel[i];
        v.x = __fmaf_rn(kk.kick, a.fx, v.x);
        v.y = __fmaf_rn(kk.kick, a.fy, v.y);
        v.z = __fmaf_rn(kk.kick, a.fz, v.z);
        kk.vel[i] = v;
        ke = kk.ke_scale * (v.x * v.x + v.y * v.y + v.z * v.z);
    }
    // per-replica fp64 reductions
    const int r0 = __shfl_sync(0xffffffffu, r, 0);
    const bool uniform = __all_sync(0xffffffffu, r == r0);
    if (e_rep) replica_add(e_rep, 1, 0, r, uniform, active, (double)ei, lane);
    if (KICK && kk.ekin) replica_add(kk.ekin, 1, 0, r, uniform, active, (double)ke, lane);
    if (VIRIAL) {
        replica_add(w_rep, 6, 0, r, uniform, active, 0.5 * (double)a.wxx, lane);
        replica_add(w_rep, 6, 1, r, uniform, active, 0.5 * (double)a.wyy, lane);
        replica_add(w_rep, 6, 2, r, uniform, active, 0.5 * (double)a.wzz, lane);
        replica_add(w_rep, 6, 3, r, uniform, active, 0.5 * (double)a.wxy, lane);
        replica_add(w_rep, 6, 4, r, uniform, active, 0.5 * (double)a.wxz, lane);
        replica_add(w_rep, 6, 5, r, uniform, active, 0.5 * (double)a.wyz, lane);
    }
}

template <bool PERIODIC>
__global__ void k_count_pairs(const float4 *__restrict__ pos, const int *__restrict__ nlist,
                              const int *__restrict__ nn, const int *__restrict__ atom_rep,
                              const RepGeom *__restrict__ geom, unsigned long long *__restrict__ out,
                              int n, int n_pad /* rows of capacity per atom */, float rc2)
{
    unsigned long long entries = 0, inside = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) {
        const float4 pi = pos[i];
        const int cnt = nn[i] & 0xffff;
        Box3 b = {0.f, 0.f, 0.f, 0};
        if (PERIODIC) {
            const RepGeom *g = geom + atom_rep[i];
            b.Lx = g->len[0]; b.Ly = g->len[1]; b.Lz = g->len[2]; b.per = g->periodic;
        }
        entries += cnt;
        for (int k = 0; k < cnt; ++k) {
            const float4 pj = pos[nlist[(tbsma_lrow(i, n_pad) + (size_t)(k >> 2) * TBSMA_LROW) * 4 + (k & 3)]];
            float dx = pi.x - pj.x, dy = pi.y - pj.y, dz = pi.z - pj.z;
            min_image<PERIODIC>(dx, dy, dz, b);
            const float d2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            inside += d2 < rc2;
        }
    }
    atomicAdd(out, entries);
    atomicAdd(out + 1, inside);
}

}  // namespace

cudaError_t tbsma_launch_density(tbsma_ctx *c, const float4 *pos, cudaStream_t st)
{
    const int n = (int)c->n;
    const int grid = (n + kBlock - 1) / kBlock;
    const int4 *nl = reinterpret_cast<const int4 *>(c->d_nlist);
    if (c->any_periodic)
        k_density<true><<<grid, kBlock, 0, st>>>(pos, nl, c->d_nn, c->d_atom_rep, c->d_geom, c->d_xs, n, c->kmax / 4, c->pc);
    else
        k_density<false><<<grid, kBlock, 0, st>>>(pos, nl, c->d_nn, c->d_atom_rep, c->d_geom, c->d_xs, n, c->kmax / 4, c->pc);
    c->launches++;
    return cudaGetLastError();
}

template <bool PERIODIC, bool VIRIAL>
static void launch_force_k(tbsma_ctx *c, float4 *force, double *e_rep, double *w_rep, KickArgs kk, cudaStream_t st)
{
    const int n = (int)c->n;
    const int grid = (n + kBlock - 1) / kBlock;
    const int4 *nl = reinterpret_cast<const int4 *>(c->d_nlist);
    if (kk.vel)
        k_force<PERIODIC, VIRIAL, true><<<grid, kBlock, 0, st>>>(c->d_xs, nl, c->d_nn, c->d_atom_rep, c->d_geom, force,
                                                                 e_rep, w_rep, kk, c->d_ctrl, n, c->kmax / 4, c->pc);
    else
        k_force<PERIODIC, VIRIAL, false><<<grid, kBlock, 0, st>>>(c->d_xs, nl, c->d_nn, c->d_atom_rep, c->d_geom, force,
                                                                  e_rep, w_rep, kk, c->d_ctrl, n, c->kmax / 4, c->pc);
}

cudaError_t tbsma_launch_force(tbsma_ctx *c, float4 *force, double *e_rep, double *w_rep, KickArgs kk,
                               cudaStream_t st)
{
    if (c->any_periodic) {
        if (w_rep) launch_force_k<true, true>(c, force, e_rep, w_rep, kk, st);
        else launch_force_k<true, false>(c, force, e_rep, w_rep, kk, st);
    } else {
        if (w_rep) launch_force_k<false, true>(c, force, e_rep, w_rep, kk, st);
        else launch_force_k<false, false>(c, force, e_rep, w_rep, kk, st);
    }
    c->launches++;
    return cudaGetLastError();
}

cudaError_t tbsma_launch_count_pairs(tbsma_ctx *c, const float4 *pos, unsigned long long *d_out2, cudaStream_t st)
{
    const int n = (int)c->n;
    int grid = (n + 255) / 256;
    if (grid > c->n_sm * 8) grid = c->n_sm * 8;
    if (c->any_periodic)
        k_count_pairs<true><<<grid, 256, 0, st>>>(pos, c->d_nlist, c->d_nn, c->d_atom_rep, c->d_geom, d_out2, n, c->kmax / 4, c->pc.rc2);
    else
        k_count_pairs<false><<<grid, 256, 0, st>>>(pos, c->d_nlist, c->d_nn, c->d_atom_rep, c->d_geom, d_out2, n, c->kmax / 4, c->pc.rc2);
    c->launches++;
    return cudaGetLastError();
}
