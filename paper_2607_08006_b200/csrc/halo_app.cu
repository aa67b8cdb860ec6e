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
        const size_t z = c % B, y = (c / B) % B, x = c / ((size_t)B * B);
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
    if (!w || w->npes != 8 || B == 0) return SHMEMG_ERR_ARG;
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
