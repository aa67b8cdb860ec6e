// halo_app.cu -- application-side kernels of the halo workload (include/shmemg_app.h).  Not library ops.
#include "internal.cuh"
#include "../../include/shmemg_app.h"

__device__ __forceinline__ unsigned long long fin64(unsigned long long x) {
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 27; x *= 0x94D049BB133111EBull;
    x ^= x >> 31;
    return x;
}
__device__ __forceinline__ unsigned long long mix64(unsigned long long seed, unsigned long long stream, unsigned long long i) {
    unsigned long long x = fin64(seed * 0xD1342543DE82EF95ull + stream * 0x9E3779B97F4A7C15ull + 0x2545F4914F6CDD1Dull);
    return fin64(x ^ (i * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull));
}

__global__ void k_halo_perturb(uint8_t *base, size_t stride, uint64_t U_off, unsigned B, unsigned long long seed,
                               unsigned long long round) {
    const int p = blockIdx.y;
    const unsigned px = (p >> 2) & 1, py = (p >> 1) & 1, pz = p & 1;
    double *U = reinterpret_cast<double *>(base + (size_t)p * stride + U_off);
    const size_t n = (size_t)B * B * B, G = 2ull * B;
    for (size_t c = (size_t)blockIdx.x * blockDim.x + threadIdx.x; c < n; c += (size_t)gridDim.x * blockDim.x) {
        const unsigned c32 = (unsigned)c, t = c32 / B, z = c32 - t * B, x = t / B, y = t - x * B;      // B^3 < 2^32 (host check)
        const size_t g = ((px * (size_t)B + x) * G + (py * (size_t)B + y)) * G + (pz * (size_t)B + z);
        U[c] = U[c] + (double)(mix64(seed, round, g) & 0xFFFFull) * 0x1.0p-30;
    }
}

__global__ void k_halo_pack(uint8_t *base, size_t stride, uint64_t send_off, uint64_t U_off, unsigned B) {
    const int p = blockIdx.z, f = blockIdx.y;
    const int axis = f >> 1, dir = f & 1;
    const double *U = reinterpret_cast<const double *>(base + (size_t)p * stride + U_off);
    double *send = reinterpret_cast<double *>(base + (size_t)p * stride + send_off) + (size_t)f * B * B;
    const size_t fix = dir ? B - 1 : 0, nn = (size_t)B * B;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < nn; k += (size_t)gridDim.x * blockDim.x) {
        const size_t a = k / B, b = k % B;
        size_t x, y, z;
        if (axis == 0) { x = fix; y = a; z = b; }
        else if (axis == 1) { x = a; y = fix; z = b; }
        else { x = a; y = b; z = fix; }
        send[k] = U[(x * B + y) * B + z];
    }
}

__global__ void k_checksum_zero(unsigned long long *out, size_t n) {
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = 0;
}
__global__ void k_checksum64(const uint8_t *base, size_t stride, uint64_t sym_off, uint64_t seg_bytes, unsigned nseg,
                             unsigned long long *out) {
    const unsigned p = blockIdx.z, s = blockIdx.y;
    const unsigned long long *x =
        reinterpret_cast<const unsigned long long *>(base + (size_t)p * stride + sym_off + (size_t)s * seg_bytes);
    const size_t n = seg_bytes >> 3;
    unsigned long long acc = 0;
    for (size_t k = (size_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (size_t)gridDim.x * blockDim.x)
        acc += __ldcg(x + k) * (2ull * k + 1ull);
    for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
    if ((threadIdx.x & 31) == 0 && acc) atomicAdd(out + (size_t)p * nseg + s, acc);
}

extern "C" int shmemg_app_halo_perturb_on_stream(shmemg_world_t *w, uint64_t U_off, uint32_t B, uint64_t seed,
                                                 uint64_t round, void *stream) {
    if (!w || w->npes != 8 || B == 0 || B > 1024) return SHMEMG_ERR_ARG;
    if (!shmemg_in_range(w, U_off, (uint64_t)B * B * B * 8)) return SHMEMG_ERR_RANGE;
    if (U_off & 7) return SHMEMG_ERR_ALIGN;
    const size_t n = (size_t)B * B * B;
    unsigned bx = (unsigned)((n + 255) / 256);
    if (bx > 148u * 16u) bx = 148u * 16u;
    k_halo_perturb<<<dim3(bx, 8), 256, 0, (cudaStream_t)stream>>>(w->base, w->stride, U_off, B, seed, round);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}
extern "C" int shmemg_app_halo_pack_on_stream(shmemg_world_t *w, uint64_t send_off, uint64_t U_off, uint32_t B,
                                              void *stream) {
    if (!w || w->npes != 8 || B == 0) return SHMEMG_ERR_ARG;
    if (!shmemg_in_range(w, U_off, (uint64_t)B * B * B * 8) || !shmemg_in_range(w, send_off, 6ull * B * B * 8))
        return SHMEMG_ERR_RANGE;
    if ((U_off | send_off) & 7) return SHMEMG_ERR_ALIGN;
    unsigned bx = (unsigned)(((size_t)B * B + 255) / 256);
    if (bx > 64) bx = 64;
    k_halo_pack<<<dim3(bx, 6, 8), 256, 0, (cudaStream_t)stream>>>(w->base, w->stride, send_off, U_off, B);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}
extern "C" int shmemg_app_checksum64_on_stream(shmemg_world_t *w, uint64_t *out, uint64_t sym_off, uint64_t seg_bytes,
                                               uint32_t nseg, void *stream) {
    if (!w || !out || nseg == 0 || nseg > 65535 || w->npes > 65535) return SHMEMG_ERR_ARG;
    if (!shmemg_in_range(w, sym_off, seg_bytes * nseg)) return SHMEMG_ERR_RANGE;
    if ((sym_off | seg_bytes) & 7) return SHMEMG_ERR_ALIGN;
    const size_t tot = (size_t)w->npes * nseg;
    k_checksum_zero<<<(unsigned)((tot + 255) / 256), 256, 0, (cudaStream_t)stream>>>((unsigned long long *)out, tot);
    unsigned bx = (unsigned)(((seg_bytes >> 3) + 256 * 8 - 1) / (256 * 8));
    if (bx == 0) bx = 1;
    if (bx > 32) bx = 32;
    k_checksum64<<<dim3(bx, nseg, w->npes), 256, 0, (cudaStream_t)stream>>>(w->base, w->stride, sym_off, seg_bytes, nseg,
                                                                          (unsigned long long *)out);
    SHMEMG_CUDA(w, cudaGetLastError());
    return SHMEMG_OK;
}

// ---- the same application, device-initiated and persistent (include/shmemg_app.h) -----------------------------------------
#include "../../include/shmemg_device.cuh"

__device__ __forceinline__ void halo_perturb_cell(double *U, size_t c, unsigned B, unsigned px, unsigned py, unsigned pz,
                                                  unsigned long long seed, unsigned long long round) {
    const unsigned c32 = (unsigned)c, t = c32 / B, z = c32 - t * B, x = t / B, y = t - x * B;          // B^3 < 2^32 (host check)
    const size_t G = 2ull * B;
    const size_t g = ((px * (size_t)B + x) * G + (py * (size_t)B + y)) * G + (pz * (size_t)B + z);
    U[c] = U[c] + (double)(mix64(seed, round, g) & 0xFFFFull) * 0x1.0p-30;
}
// all blocks of one PE's group: arrive (release) and wait until the whole group has (acquire); counters are monotonic
__device__ __forceinline__ void halo_group_sync(unsigned *bar, unsigned group) {
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned old;
        asm volatile("atom.acq_rel.gpu.global.add.u32 %0, [%1], 1;" : "=r"(old) : "l"(bar) : "memory");
        const unsigned target = (old / group + 1u) * group;
        unsigned v;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory"); } while ((int)(v - target) < 0);
    }
    __syncthreads();
}

// Roles inside one PE's group of blocks:
//   blocks 0..5 ("face blocks")  per round: perturb the boundary cells they own (x-planes: blocks 0,1; y-planes without the
//                x-planes: 2,3; z-planes without both: 4,5); the six synchronise (every face plane is final); block f puts face
//                f straight out of the cube into the neighbour's ghost[round & 1] and signals; then waits for its own incoming
//                face of this round.
//   blocks 6..   ("interior blocks") perturb the interior, one warp per row, and never synchronise with anybody inside the
//                round; before the next round they check that this round's six faces have arrived (the dependency a stencil
//                would have on its ghost cells; long satisfied by then).
__global__ void __launch_bounds__(512) k_halo_persistent(const shmemg_device_world_t dw, unsigned *group_bar, uint64_t U_off,
                                                         uint64_t ghost_off, uint64_t sig_off, unsigned B, unsigned long long seed,
                                                         unsigned long long first_round, unsigned rounds, unsigned group) {
    const unsigned p = blockIdx.x / group, g = blockIdx.x % group;           // PE and block within the PE's group
    const unsigned px = (p >> 2) & 1, py = (p >> 1) & 1, pz = p & 1;
    double *U = reinterpret_cast<double *>(shmemg_dev_ptr(dw, U_off, (int)p));
    const size_t fb = (size_t)B * B * 8;
    if (g < 6) {
        const unsigned f = g, axis = f >> 1, dir = f & 1, t = p ^ (4u >> axis), fr = 2 * axis + (1 - dir);
        const size_t fix = dir ? B - 1 : 0;
        for (unsigned long long r = first_round; r < first_round + rounds; ++r) {
            // (a) the boundary cells this block owns, each cell of the cube's surface exactly once over the six blocks
            const size_t cnt = axis == 0 ? (size_t)B * B : axis == 1 ? (B > 2 ? (size_t)(B - 2) * B : 0)
                                                                     : (B > 2 ? (size_t)(B - 2) * (B - 2) : 0);
            for (size_t k = threadIdx.x; k < cnt; k += blockDim.x) {
                size_t x, y, z;
                if (axis == 0) { x = fix; y = k / B; z = k % B; }
                else if (axis == 1) { x = 1 + k / B; y = fix; z = k % B; }
                else { x = 1 + k / (B - 2); y = 1 + k % (B - 2); z = fix; }
                if (B == 1 && dir == 1) continue;                             // B = 1: the single cell belongs to face 0
                halo_perturb_cell(U, (x * B + y) * B + z, B, px, py, pz, seed, r);
            }
            __threadfence();
            halo_group_sync(group_bar + p, 6);                                // all six face planes of this PE are final
            // (b) face f = 2*axis + dir lands in slot 2*axis + (1-dir) of the neighbour along axis
            const uint64_t dst = ghost_off + (((r & 1) * 6 + fr) * fb);
            if (axis == 0) shmemg_dev_ibput_block(dw, dst, U_off + fix * fb, 0, 0, fb, 1, (int)p, (int)t);
            else if (axis == 1) shmemg_dev_ibput_block(dw, dst, U_off + fix * B * 8, (uint64_t)B * 8, fb, (size_t)B * 8, B, (int)p, (int)t);
            else shmemg_dev_ibput_block(dw, dst, U_off + fix * 8, 8, (uint64_t)B * 8, 8, (size_t)B * B, (int)p, (int)t);
            shmemg_dev_signal_block(dw, sig_off + fr * 8, r, SHMEMG_SIGNAL_SET, (int)t);
            // (c) my own incoming face of this round (keeps neighbours within one round of each other)
            shmemg_dev_signal_wait_until_block(dw, sig_off + f * 8, SHMEMG_CMP_GE, r, (int)p);
            halo_group_sync(group_bar + p, 6);                                // nobody perturbs a plane that is still being read
        }
        return;
    }
    // interior blocks: one warp per interior row (x, y): no division per cell, coalesced, eight independent cells per lane
    const unsigned lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const size_t gw = (size_t)(g - 6) * wpb + (threadIdx.x >> 5), GW = (size_t)(group - 6) * wpb;
    for (unsigned long long r = first_round; r < first_round + rounds; ++r) {
        for (size_t row = gw; row < (size_t)B * B; row += GW) {
            const unsigned x = (unsigned)(row / B), y = (unsigned)(row - (size_t)x * B);
            if (x == 0 || x == B - 1 || y == 0 || y == B - 1) continue;
            double *Ur = U + row * B;
            const size_t g0 = ((px * (size_t)B + x) * (2ull * B) + (py * (size_t)B + y)) * (2ull * B) + pz * (size_t)B;
            for (unsigned z0 = lane; z0 < B; z0 += 256) {
                double v[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const unsigned z = z0 + 32u * u;
                    if (z > 0 && z < B - 1) v[u] = Ur[z];
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const unsigned z = z0 + 32u * u;
                    if (z > 0 && z < B - 1) Ur[z] = v[u] + (double)(mix64(seed, r, g0 + z) & 0xFFFFull) * 0x1.0p-30;
                }
            }
        }
        if (threadIdx.x < 6) shmemg_dev_signal_wait_until(dw, sig_off + threadIdx.x * 8, SHMEMG_CMP_GE, r, (int)p);
        __syncthreads();
    }
}

extern "C" int shmemg_app_halo_persistent_on_stream(shmemg_world_t *w, uint64_t U_off, uint64_t ghost_off, uint64_t sig_off,
                                                    uint32_t B, uint64_t seed, uint64_t first_round, uint32_t rounds,
                                                    void *stream) {
    if (!w || w->npes != 8 || B == 0 || B > 1024) return SHMEMG_ERR_ARG;
    const uint64_t fb = (uint64_t)B * B * 8;
    if (!shmemg_in_range(w, U_off, fb * B) || !shmemg_in_range(w, ghost_off, 12 * fb) || !shmemg_in_range(w, sig_off, 48))
        return SHMEMG_ERR_RANGE;
    if ((U_off | ghost_off | sig_off) & 7) return SHMEMG_ERR_ALIGN;
    if (rounds == 0) return SHMEMG_OK;
    int per_sm = 0;
    SHMEMG_CUDA(w, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_halo_persistent, 512, 0));
    unsigned group = (unsigned)((size_t)w->sm_count * per_sm / 8);
    if (group < 7) return SHMEMG_ERR_NOMEM;                                   // six face blocks + interior blocks per PE, all co-resident
    if (group > 64) group = 64;
    shmemg_device_world_t dw;
    int rc = shmemg_device_world_get(w, &dw);
    if (rc) return rc;
    unsigned *bar = w->ctl->group_bar;
    unsigned long long seed_ = seed, first_ = first_round;
    void *args[] = {&dw, &bar, &U_off, &ghost_off, &sig_off, &B, &seed_, &first_, &rounds, &group};
    SHMEMG_CUDA(w, cudaLaunchCooperativeKernel((void *)k_halo_persistent, dim3(8 * group), dim3(512), args, 0, (cudaStream_t)stream));
    return SHMEMG_OK;
}
