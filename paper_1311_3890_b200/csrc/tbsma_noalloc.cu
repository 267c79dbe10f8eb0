// tbsma_noalloc.cu -- tbsma_kinetic_tensor_noalloc: the kinetic tensor K_ab = sum_i m v_i,a v_i,b of every replica
// (Eq.5 as read in D:A11) for callers that must not allocate device memory.
//
// Who that is.  Every other entry point of this library works through a tbsma_ctx, and tbsma_set_system /
// tbsma_build_cells call cudaMalloc for the context's tables.  Some hosts of this code cannot afford that, or are not
// allowed to:
//   - an MD engine or a training framework that took (nearly) all of the GPU's memory into its own pool at start-up:
//     a cudaMalloc from a plug-in then fails, or succeeds by taking memory the pool's owner believes it has;
//   - a loop that must not stall: cudaMalloc and cudaFree synchronise the whole device, so one call from an analysis
//     hook between two MD steps drains every stream of the process;
//   - a process under a fixed memory budget (several jobs sharing one GPU), where every byte is accounted for before
//     the run starts.
// Such a caller owns pos / vel / offsets / the output, as always, and this file brings the only other memory the
// kernel needs with it: a fixed array in the library's device image.
//
// The kernel is a variant of k_kinetic_tensor (tbsma_integrate.cu).  That one looks the replica of each atom up in a
// per-atom table of the context (c->d_atom_rep, allocated by tbsma_set_system) and adds with fp64 atomics.  This one
// needs no per-atom table: a CTA is given (replica, slice) by its block index, sums its slice of the replica's atoms in
// a fixed order, writes six partial sums to the scratch array, and the last CTA of a replica to finish (a ticket
// counter in the same array) adds the replica's partial sums in slice order.  The sums are therefore also bitwise
// repeatable, which the atomic version is not.
//
// The scratch array
//   static __device__ __align__(256) unsigned char g_scratch[TBSMA_NOALLOC_SCRATCH_BYTES]   (784 KiB)
//     [0, 16 KiB)         one 32-bit ticket per replica   (TBSMA_NOALLOC_MAX_REPLICAS = 4096)
//     [16 KiB, 784 KiB)   six doubles per (replica, slice) (TBSMA_NOALLOC_MAX_SLOTS = 16384)
// lives in every GPU that loads libtbsma.so, from the moment the CUDA runtime loads the library's device code on that
// GPU until the process exits, whether or not this entry point is ever called.  It is ONE array per GPU: every call on
// that GPU, from any thread or stream, uses it.  Two calls that may run on the GPU at the same time (different
// streams, no dependency between them) race on the tickets and the partial sums and both results are garbage; issue
// the calls on one stream, or order them with events.  The array also keeps whatever the previous call left in it.
// The partial sums are all written before they are read, so stale ones do no harm; the tickets must start at zero, and
// every call clears the tickets it is going to use first (a cudaMemsetAsync on the caller's stream, which allocates
// nothing), so a call that was cut short by an error cannot poison the next one.
//
// Host code cannot use the name g_scratch as a pointer: on the host that name is only a handle by which the runtime
// finds the device array, and a kernel handed &g_scratch[0] from host code would read host address space.  The
// device address is asked for once per GPU with cudaGetSymbolAddress, with that GPU current, and cached below.  The
// FIRST call of tbsma_kinetic_tensor_noalloc on a GPU does this set-up (it may also make the runtime load the library's
// device code, which takes a while); make that first call before starting any stream capture.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "tbsma_internal.cuh"

#define NOALLOC_THREADS 256
#define NOALLOC_TICKET_BYTES (TBSMA_NOALLOC_MAX_REPLICAS * 4)
#define NOALLOC_SCRATCH_BYTES (NOALLOC_TICKET_BYTES + TBSMA_NOALLOC_MAX_SLOTS * 6 * 8)
#define NOALLOC_MAX_DEVICES 64

static_assert(NOALLOC_SCRATCH_BYTES == TBSMA_NOALLOC_SCRATCH_BYTES, "tbsma.h states the size of the scratch array");
static_assert(NOALLOC_TICKET_BYTES % 256 == 0, "the partial sums start on a 256-byte boundary");

static __device__ __align__(256) unsigned char g_scratch[NOALLOC_SCRATCH_BYTES];

namespace {

// CTA (s, r) of a grid of S x R: atoms [b + len s / S, b + len (s + 1) / S) of replica r = [b, b + len).
// Order of every sum: thread-strided over the slice, a shuffle tree over the 32 lanes, the 8 warps in order, the S
// slices in order.  It depends on (offsets, S) only.
__global__ void __launch_bounds__(NOALLOC_THREADS)
k_kinetic_tensor_sliced(const float4 *__restrict__ pos, const float4 *__restrict__ vel, const int *__restrict__ off,
                        unsigned char *scratch, double *__restrict__ k_rep, double m_over_c, int S)
{
    __shared__ double s_w[NOALLOC_THREADS / 32][6];
    __shared__ int s_last;
    unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch);
    double *part = reinterpret_cast<double *>(scratch + NOALLOC_TICKET_BYTES);
    const int s = blockIdx.x, r = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long b = off[r], len = (long long)off[r + 1] - b;
    double k[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    if (len > 0) {
        const long long i0 = b + len * s / S, i1 = b + len * (s + 1) / S;
        for (long long i = i0 + tid; i < i1; i += NOALLOC_THREADS) {
            if ((__float_as_int(pos[i].w) & 3) != 0) continue;          // grip atoms are not dynamic (D:A10)
            const float4 v = vel[i];
            const double vx = v.x, vy = v.y, vz = v.z;
            k[0] += m_over_c * vx * vx; k[1] += m_over_c * vy * vy; k[2] += m_over_c * vz * vz;
            k[3] += m_over_c * vx * vy; k[4] += m_over_c * vx * vz; k[5] += m_over_c * vy * vz;
        }
    }
#pragma unroll
    for (int c = 0; c < 6; ++c) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) k[c] += __shfl_xor_sync(0xffffffffu, k[c], o);
        if (lane == 0) s_w[warp][c] = k[c];
    }
    __syncthreads();
    if (tid < 6) {
        double a = 0.0;
#pragma unroll
        for (int w = 0; w < NOALLOC_THREADS / 32; ++w) a += s_w[w][tid];
        __stcg(part + 6 * ((size_t)r * S + s) + tid, a);
        __threadfence();                                                 // the partial sum is visible before the ticket
    }
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        s_last = atomicAdd(ticket + r, 1u) == (unsigned int)(S - 1);
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    if (tid < 6) {
        double a = 0.0;
        for (int q = 0; q < S; ++q) a += __ldcg(part + 6 * ((size_t)r * S + q) + tid);
        k_rep[6 * (size_t)r + tid] = a;
    }
}

std::mutex g_mu;
unsigned char *g_scratch_of[NOALLOC_MAX_DEVICES];     // device address of g_scratch on GPU d, nullptr until asked for

// Device address of the scratch array on the CURRENT device; asks the runtime the first time, then answers from the
// cache.  Nothing is allocated: the array is part of the library's device image.
cudaError_t scratch_of_current_device(unsigned char **out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_of[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_of[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_of[dev];
    return cudaSuccess;
}

}  // namespace

extern "C" int tbsma_kinetic_tensor_noalloc(const float *d_pos, const float *d_vel, const int32_t *d_replica_offsets,
                                            int64_t n_atoms, int32_t n_replicas, double mass_amu,
                                            double *d_replica_kinetic, void *stream)
{
    if (n_atoms < 0 || n_replicas < 0 || !(mass_amu > 0.0)) return TBSMA_EINVAL;
    if (n_replicas > TBSMA_NOALLOC_MAX_REPLICAS || n_atoms > TBSMA_NOALLOC_MAX_ATOMS) return TBSMA_ELIMIT;
    if (n_replicas == 0) return TBSMA_OK;
    if (!d_replica_offsets || !d_replica_kinetic || (n_atoms > 0 && (!d_pos || !d_vel))) return TBSMA_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    unsigned char *scratch = nullptr;
    cudaError_t e = scratch_of_current_device(&scratch);
    if (e != cudaSuccess) return TBSMA_ECUDA;
    // slices per replica: about 1024 atoms each, at most 256, and no more than the partial-sum slots allow
    const int64_t per_rep = n_atoms / n_replicas;
    int64_t S = (per_rep + 1023) / 1024;
    const int64_t s_cap = TBSMA_NOALLOC_MAX_SLOTS / n_replicas;
    if (S > 256) S = 256;
    if (S > s_cap) S = s_cap;
    if (S < 1) S = 1;
    e = cudaMemsetAsync(scratch, 0, sizeof(unsigned int) * (size_t)n_replicas, st);      // tickets start at zero
    if (e != cudaSuccess) return TBSMA_ECUDA;
    k_kinetic_tensor_sliced<<<dim3((unsigned)S, (unsigned)n_replicas), NOALLOC_THREADS, 0, st>>>(
        reinterpret_cast<const float4 *>(d_pos), reinterpret_cast<const float4 *>(d_vel), d_replica_offsets, scratch,
        d_replica_kinetic, mass_amu / TBSMA_ACC, (int)S);
    return cudaGetLastError() == cudaSuccess ? TBSMA_OK : TBSMA_ECUDA;
}
