/*
 * cs_recount.cu -- second pass over the stream restricted to a set of output cells:
 *   - exact recount: counts[i] += number of particles whose cell is ids[i]          ("the exact
 *     number of particles in the output cells", used to estimate the false-positive rate);
 *   - membership filter: the particles of those cells are copied out densely           (Fig. 14:
 *     keep the particles of the heavy cells and hand them to an offline halo finder).
 * The id set is held as an open-addressing hash table (load factor <= 1/4) built on the device per call.
 */
#include "cs_device.cuh"
#include "cs_launch.cuh"

namespace cs {

constexpr uint64_t HT_EMPTY = ~0ull;

__device__ __forceinline__ uint32_t ht_slot(uint64_t c, uint32_t mask) { return (uint32_t)(mix64(c ^ 0x6A09E667F3BCC909ULL) >> 20) & mask; }

__global__ void __launch_bounds__(256)
k_ht_build(const uint64_t* __restrict__ ids, uint32_t m, unsigned long long* __restrict__ keys, uint32_t* __restrict__ vals,
           uint32_t mask) {
    const uint32_t i = blockIdx.x * 256 + threadIdx.x;
    if (i >= m) return;
    const uint64_t c = ids[i];
    uint32_t s = ht_slot(c, mask);
    for (;;) {
        const unsigned long long old = atomicCAS(&keys[s], (unsigned long long)HT_EMPTY, (unsigned long long)c);
        if (old == HT_EMPTY || old == c) { atomicMin(&vals[s], i); return; }   // vals start at ~0u; duplicate id: the first occurrence counts
        s = (s + 1) & mask;
    }
}

/* index of c in ids, or ~0u */
__device__ __forceinline__ uint32_t ht_find(const unsigned long long* __restrict__ keys, const uint32_t* __restrict__ vals,
                                            uint32_t mask, uint64_t c) {
    uint32_t s = ht_slot(c, mask);
    for (;;) {
        const unsigned long long k = keys[s];
        if (k == c) return vals[s];
        if (k == HT_EMPTY) return ~0u;
        s = (s + 1) & mask;
    }
}

__device__ __forceinline__ void recount_particle(const ScaleParams& sp, const unsigned long long* keys, const uint32_t* vals,
                                                 uint32_t mask, uint32_t* counts, float* out, uint32_t* out_count,
                                                 uint64_t cap, bool in, float x, float y, float z) {
    bool hit = false;
    if (in) {
        const uint32_t idx = ht_find(keys, vals, mask, cell_of(x, y, z, sp));
        hit = idx != ~0u;
        if (hit) atomicAdd(&counts[idx], 1u);
    }
    const uint32_t m = __ballot_sync(0xFFFFFFFFu, hit);
    if (m == 0) return;
    const uint32_t lane = threadIdx.x & 31u;
    const int leader = __ffs(m) - 1;
    uint32_t base = 0;
    if ((int)lane == leader) base = atomicAdd(out_count, (uint32_t)__popc(m));
    base = __shfl_sync(0xFFFFFFFFu, base, leader);
    if (hit) {
        const uint64_t at = (uint64_t)base + __popc(m & ((1u << lane) - 1u));
        if (out && at < cap) { out[3 * at] = x; out[3 * at + 1] = y; out[3 * at + 2] = z; }
    }
}

__global__ void __launch_bounds__(PASS_THREADS)
k_recount(const __grid_constant__ ScaleParams sp, const float* __restrict__ xyz, uint64_t n, uint32_t head, uint64_t groups,
          const unsigned long long* __restrict__ keys, const uint32_t* __restrict__ vals, uint32_t mask,
          uint32_t* __restrict__ counts, float* __restrict__ out, uint32_t* out_count, uint64_t cap) {
    const uint64_t stride = (uint64_t)gridDim.x * PASS_THREADS;
    const float4* body = reinterpret_cast<const float4*>(xyz + 3 * (uint64_t)head);
    const uint32_t lane = threadIdx.x & 31u;
    for (uint64_t g0 = (uint64_t)blockIdx.x * PASS_THREADS + (threadIdx.x - lane); g0 < groups; g0 += stride) {
        const uint64_t g = g0 + lane;
        const bool in = g < groups;
        float4 q0 = make_float4(0.f, 0.f, 0.f, 0.f), q1 = q0, q2 = q0;
        if (in) {
            q0 = ld_stream16(body + 3 * g);
            q1 = ld_stream16(body + 3 * g + 1);
            q2 = ld_stream16(body + 3 * g + 2);
        }
        recount_particle(sp, keys, vals, mask, counts, out, out_count, cap, in, q0.x, q0.y, q0.z);
        recount_particle(sp, keys, vals, mask, counts, out, out_count, cap, in, q0.w, q1.x, q1.y);
        recount_particle(sp, keys, vals, mask, counts, out, out_count, cap, in, q1.z, q1.w, q2.x);
        recount_particle(sp, keys, vals, mask, counts, out, out_count, cap, in, q2.y, q2.z, q2.w);
    }
    if (blockIdx.x == 0 && threadIdx.x < 32) {        // warp 0: the <= 6 edge particles
        const uint64_t tail0 = (uint64_t)head + 4 * groups;
        const uint64_t n_edge = (uint64_t)head + (n - tail0);
        const bool in = threadIdx.x < n_edge;
        float x = 0.f, y = 0.f, z = 0.f;
        if (in) {
            const uint64_t i = threadIdx.x < head ? threadIdx.x : tail0 + (threadIdx.x - head);
            const float* p = xyz + 3 * i;
            x = ld_stream4(p); y = ld_stream4(p + 1); z = ld_stream4(p + 2);
        }
        recount_particle(sp, keys, vals, mask, counts, out, out_count, cap, in, x, y, z);
    }
}

/* keys: table of (mask + 1) words, filled with HT_EMPTY by the caller; vals: same length */
cudaError_t launch_ht_build(const uint64_t* ids, uint32_t m, uint64_t* keys, uint32_t* vals, uint32_t mask, cudaStream_t st) {
    if (!m) return cudaSuccess;
    k_ht_build<<<(m + 255) / 256, 256, 0, st>>>(ids, m, reinterpret_cast<unsigned long long*>(keys), vals, mask);
    return cudaGetLastError();
}

cudaError_t launch_recount(const ScaleParams& sp, const float* xyz, uint64_t n, const uint64_t* keys, const uint32_t* vals,
                           uint32_t mask, uint32_t* counts, float* out, uint32_t* out_count, uint64_t cap, int sm_count,
                           cudaStream_t st) {
    uint32_t head;
    uint64_t groups;
    split_aligned(xyz, n, &head, &groups);
    int blocks = blocks_for(k_recount, sm_count, groups);
    k_recount<<<blocks, PASS_THREADS, 0, st>>>(sp, xyz, n, head, groups, reinterpret_cast<const unsigned long long*>(keys), vals,
                                               mask, counts, out, out_count, cap);
    return cudaGetLastError();
}

}  // namespace cs
