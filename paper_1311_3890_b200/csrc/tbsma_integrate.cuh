// tbsma_integrate.cuh -- device code of the opening half of the MD step, shared by
// tbsma_integrate.cu (k_integrate_pre) and tbsma_tile.cu (the fused step of small batches).  Product code.
#pragma once
#include "tbsma_internal.cuh"

// Philox4x32-10 (Salmon et al., SC'11), written out; D:A9 fixes key/counter layout:
// key = (seed_lo, seed_hi), counter = (tag inside replica, step_lo, step_hi, 0).
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k)
{
    const unsigned M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int round = 0; round < 10; ++round) {
        const unsigned hi0 = __umulhi(M0, c.x), lo0 = M0 * c.x;
        const unsigned hi1 = __umulhi(M1, c.z), lo1 = M1 * c.z;
        c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
        k.x += W0; k.y += W1;
    }
    return c;
}

// u = ((x >> 8) + 0.5) 2^-24 in (0,1); Box-Muller as in D:A9.
__device__ __forceinline__ float3 gauss3(unsigned long long seed, unsigned tag, unsigned long long step)
{
    const uint4 x = philox4x32_10(make_uint4(tag, (unsigned)step, (unsigned)(step >> 32), 0u),
                                  make_uint2((unsigned)seed, (unsigned)(seed >> 32)));
    const float s = 1.0f / 16777216.0f, h = 0.5f / 16777216.0f;
    const float u0 = __fmaf_rn((float)(x.x >> 8), s, h), u1 = __fmaf_rn((float)(x.y >> 8), s, h);
    const float u2 = __fmaf_rn((float)(x.z >> 8), s, h), u3 = __fmaf_rn((float)(x.w >> 8), s, h);
    const float ra = sqrtf(-2.0f * logf(u0)), rb = sqrtf(-2.0f * logf(u2));
    float sn, cs, cs2;
    sincospif(2.0f * u1, &sn, &cs);
    cs2 = cospif(2.0f * u3);
    return make_float3(ra * cs, ra * sn, rb * cs2);
}

// One atom (or, for i < R, also one replica's accumulators) of the opening half of the step; called by
// k_integrate_pre and by the fused step kernel of small batches (tbsma_tile.cu: k_step_small).
__device__ __forceinline__ void tbsma_integrate_one(int i, float4 *__restrict__ pos, float4 *__restrict__ vel, const float4 *__restrict__ force,
                const float4 *__restrict__ pos_build, const int *__restrict__ atom_rep,
                const RepGeom *__restrict__ geom, const int *__restrict__ tag, const StepArgs &a,
                const unsigned long long *__restrict__ counters, int *__restrict__ dirty,
                int *__restrict__ ctrl, int n, int R)
{
    if (i < R) {   // zero the per-replica accumulators of the force pass that follows
        if (a.e_rep) a.e_rep[i] = 0.0;
        if (a.ekin) a.ekin[i] = 0.0;
        if (a.w_rep) for (int k = 0; k < 6; ++k) a.w_rep[6 * i + k] = 0.0;
    }
    if (i < n) {
    const unsigned long long off = counters[0];
    const unsigned long long step = (a.step_on_device ? counters[7] : a.step_base) + off;
    const int r = atom_rep[i];
    float4 p = pos[i], v = vel[i];
    const int flag = __float_as_int(p.w) & 3;
    if (flag == 0) {
        const float4 f = force[i];
        v.x = __fmaf_rn(a.kick, f.x, v.x); v.y = __fmaf_rn(a.kick, f.y, v.y); v.z = __fmaf_rn(a.kick, f.z, v.z);
        p.x = __fmaf_rn(a.half_dt, v.x, p.x); p.y = __fmaf_rn(a.half_dt, v.y, p.y); p.z = __fmaf_rn(a.half_dt, v.z, p.z);
        if (a.nh_scale) {              // N of B A N A B (Nose-Hoover, k_nh_update): v *= exp(-xi dt)
            const float sc = a.nh_scale[r];
            v.x *= sc; v.y *= sc; v.z *= sc;
        } else if (a.thermostat) {
            const unsigned trel = (unsigned)(tag[i] - geom[r].atom_begin);
            const float3 g = gauss3(a.seed[r], trel, step);
            const float Tr = a.T_rate ? (float)((double)a.T[r] + (double)a.T_rate[r] * (double)off) : a.T[r];
            const float sg = a.c2 * a.sigma_scale * sqrtf(fmaxf(Tr, 0.f));
            v.x = __fmaf_rn(a.c1, v.x, sg * g.x); v.y = __fmaf_rn(a.c1, v.y, sg * g.y); v.z = __fmaf_rn(a.c1, v.z, sg * g.z);
        }
        p.x = __fmaf_rn(a.half_dt, v.x, p.x); p.y = __fmaf_rn(a.half_dt, v.y, p.y); p.z = __fmaf_rn(a.half_dt, v.z, p.z);
    } else {       // rigid grip atom (D:A12): v = 0; a pulled atom is placed, never incremented (D:A10)
        v.x = v.y = v.z = 0.f;
        // steps of slab motion since the run began: every step, or in strokes of `period` steps
        unsigned long long nst = off + 1ull;
        if (a.period > 0) nst = nst / (unsigned long long)a.period * (unsigned long long)a.period;
        if (flag == 2) {
            double D = a.disp0 ? a.disp0[r] : 0.0;
            if (a.rate) D += a.rate[r] * (double)nst;
            p.z = (float)((double)v.w + D);
        } else if (a.disp0_1 || a.rate_1) {      // the other end (both ends move); without a schedule it stays fixed
            double D = a.disp0_1 ? a.disp0_1[r] : 0.0;
            if (a.rate_1) D += a.rate_1[r] * (double)nst;
            p.z = (float)((double)v.w + D);
        }
    }
    pos[i] = p;
    vel[i] = v;
    const float4 pb = pos_build[(size_t)a.cur[r] * a.pb_stride + i];
    const float dx = p.x - pb.x, dy = p.y - pb.y, dz = p.z - pb.z;
    const float d2 = dx * dx + dy * dy + dz * dz;
    const bool cadence = a.rebuild_every > 0 && (step % (unsigned long long)a.rebuild_every) == 0ull;
    if (d2 > a.skin_half2 && a.trigger2 < a.skin_half2) atomicOr(ctrl + 1, (int)TBSMA_FLAG_SKIN_VIOLATED);
    // (the staggered first rebuild is for displacement-triggered lists only: with a fixed cadence an early trigger
    // would be reported as a violated skin)
    const float trig2 = a.rebuild_every > 0 ? a.trigger2 : a.trigger2 * a.stagger[r];
    if (d2 > trig2 || cadence) {
        // level 2 = cells + candidate list too (tile variant, decided at the replica's previous rebuild)
        const int level = (a.want_outer && a.want_outer[r]) ? 2 : 1;
        dirty[r] = level;
        ctrl[0] = 1;
        if (level == 2) ctrl[3] = 1;
        if (a.rebuild_every > 0 && !cadence) atomicOr(ctrl + 1, (int)TBSMA_FLAG_SKIN_VIOLATED);
    }
    }
}

