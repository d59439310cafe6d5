/*
 * aesoff_calib.cu -- calibration microkernels for the roofline of DESIGN.md section 6 (SURVEY.md
 * section 7, step 4): what the units the cipher leans on really deliver on this GPU, measured with the
 * engine's own table layout and launch shape (one CTA per SM, 16 warps, 128 KiB of replicated tables).
 *
 *   lookup   PRMT-built address + LDS.32, conflict-free by construction (lane l reads bank l), 16
 *            independent chains per thread: the shared-memory data pipe's lookup rate.
 *   alu      the same instruction mix without the loads (PRMT + LOP3): the ALU pipe's rate.
 *   round    the cipher's main round as it stands (per column 4 PRMT + 4 LDS + 2 LOP3, 4 blocks per lane):
 *            what the two pipes deliver together, i.e. the ceiling of the kernel's inner loop.
 *   copy     128-bit L2-only loads and stores of a buffer larger than L2: the payload path's HBM rate.
 *   bitslice the alternative the table form was chosen against: a bitsliced S-box
 *            (aesoff_bitslice.cuh: tower-field circuit derived and checked by gen_bitslice_sbox.py), first
 *            verified on all 256 inputs against S[x] as read out of T0, then run as 4 independent chains
 *            per thread: S-box evaluations (32 lanes x 32 bytes each) per clock per SM.
 *
 * Nothing here is on the product path; aes_calibrate() is called by bench.py and the tests only.
 */
#include <cuda_runtime.h>
#include <stdint.h>

#include "aesoff_bitslice.cuh"
#include "aesoff_cipher.cuh"
#include "aesoff_internal.h"

using namespace aesoff;

namespace {

constexpr int CALIB_THREADS = 512;
constexpr int CALIB_CHAINS = 16;

__global__ void __launch_bounds__(CALIB_THREADS, 1)
calib_lookup_kernel(const uint32_t *T0, uint32_t iters, uint32_t *sink, unsigned long long *cycles, int with_loads)
{
    extern __shared__ __align__(128) uint8_t smem[];
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem);
    const uint32_t tbase = (sbase + 65535u) & ~65535u;
    fill_tables(tbase, T0, threadIdx.x, CALIB_THREADS);
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31u, ybase = tbase | (lane * 4u);
    uint32_t x[CALIB_CHAINS];
#pragma unroll
    for (int i = 0; i < CALIB_CHAINS; ++i) x[i] = (threadIdx.x * 2654435761u) ^ (i * 0x9e3779b9u) ^ blockIdx.x;
    unsigned long long g0, g1;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
    const long long t0 = clock64();
    for (uint32_t it = 0; it < iters; ++it) {
        if (with_loads == 2) {
            /* the cipher's main round as it stands (4 blocks per lane, no round-key loads): per column
             * 4 PRMT + 4 LDS + 2 LOP3 */
#pragma unroll
            for (int i = 0; i < CALIB_CHAINS; i += 4) {
                const uint32_t x0 = x[i + 0], x1 = x[i + 1], x2 = x[i + 2], x3 = x[i + 3];
                x[i + 0] = TL(0, 0, x0) ^ TL(1, 1, x1) ^ TL(2, 2, x2) ^ TL(3, 3, x3) ^ it;
                x[i + 1] = TL(0, 0, x1) ^ TL(1, 1, x2) ^ TL(2, 2, x3) ^ TL(3, 3, x0) ^ it;
                x[i + 2] = TL(0, 0, x2) ^ TL(1, 1, x3) ^ TL(2, 2, x0) ^ TL(3, 3, x1) ^ it;
                x[i + 3] = TL(0, 0, x3) ^ TL(1, 1, x0) ^ TL(2, 2, x1) ^ TL(3, 3, x2) ^ it;
            }
        } else if (with_loads) {
#pragma unroll
            for (int i = 0; i < CALIB_CHAINS; i += 4) { /* the cipher's own pattern: four tables, four byte positions */
                x[i + 0] = TL(0, 0, x[i + 0]);
                x[i + 1] = TL(1, 1, x[i + 1]);
                x[i + 2] = TL(2, 2, x[i + 2]);
                x[i + 3] = TL(3, 3, x[i + 3]);
            }
        } else {
#pragma unroll
            for (int i = 0; i < CALIB_CHAINS; i += 4) { /* address build + a three-input XOR, no load */
                const uint32_t a = taddr<0>(x[i + 0], ybase), b = taddr<1>(x[i + 1], ybase);
                const uint32_t c = taddr<2>(x[i + 2], ybase), d = taddr<3>(x[i + 3], ybase);
                x[i + 0] = a ^ b ^ x[i + 2];
                x[i + 1] = b ^ c ^ x[i + 3];
                x[i + 2] = c ^ d ^ x[i + 0];
                x[i + 3] = d ^ a ^ x[i + 1];
            }
        }
    }
    const long long t1 = clock64();
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
    uint32_t acc = 0;
#pragma unroll
    for (int i = 0; i < CALIB_CHAINS; ++i) acc ^= x[i];
    if (acc == 0x12345678u) sink[0] = acc; /* keeps the chains alive */
    if (threadIdx.x == 0) {
        cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
        cycles[gridDim.x + blockIdx.x] = g1 - g0; /* nanoseconds of the same interval: the SM clock is their ratio */
    }
}

constexpr int BS_CHAINS = 4;
__global__ void __launch_bounds__(CALIB_THREADS, 1)
calib_bitslice_kernel(const uint32_t *T0, uint32_t iters, uint32_t *sink, unsigned long long *cycles, uint32_t *mismatches)
{
    /* correctness first: pass p covers the byte values 32 p + j, j = lane-independent bit position */
    if (blockIdx.x == 0 && threadIdx.x < 8) {
        const uint32_t p = threadIdx.x;
        uint32_t x[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            x[k] = 0;
            for (uint32_t j = 0; j < 32; ++j) x[k] |= (((32u * p + j) >> k) & 1u) << j;
        }
        bitslice_sbox(x);
        uint32_t bad = 0;
        for (uint32_t j = 0; j < 32; ++j) {
            uint32_t s = 0;
#pragma unroll
            for (int k = 0; k < 8; ++k) s |= ((x[k] >> j) & 1u) << k;
            if (s != ((__ldg(T0 + 32u * p + j) >> 8) & 0xffu)) ++bad; /* byte 1 of T0[v] is S[v] */
        }
        if (bad) atomicAdd(mismatches, bad);
    }
    uint32_t st[BS_CHAINS][8];
#pragma unroll
    for (int c = 0; c < BS_CHAINS; ++c)
#pragma unroll
        for (int k = 0; k < 8; ++k) st[c][k] = (threadIdx.x * 2654435761u) ^ ((c * 8 + k) * 0x9e3779b9u) ^ blockIdx.x;
    __syncthreads();
    const long long t0 = clock64();
    for (uint32_t it = 0; it < iters; ++it) {
#pragma unroll
        for (int c = 0; c < BS_CHAINS; ++c) bitslice_sbox(st[c]);
    }
    const long long t1 = clock64();
    uint32_t acc = 0;
#pragma unroll
    for (int c = 0; c < BS_CHAINS; ++c)
#pragma unroll
        for (int k = 0; k < 8; ++k) acc ^= st[c][k];
    if (acc == 0x12345678u) sink[0] = acc;
    if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
}

__global__ void __launch_bounds__(CALIB_THREADS, 2) calib_copy_kernel(const uint4 *src, uint4 *dst, size_t n16)
{
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n16; i += stride) __stcg(dst + i, __ldcg(src + i));
}

} /* namespace */

/* Fills out[0..5]: lookups per clock per SM, ALU instructions (warp-wide) per clock per SM, copy GB/s
 * (read + write bytes), SM clock in MHz during the lookup run, SM count, lookups per clock per SM of the
 * cipher's own main-round instruction mix.  Returns 0 or a CUDA error.                                   */
extern "C" int aesoff_run_calibration(int device, double out[8])
{
    AesoffDeviceScope on_device(device); /* the caller's current device is restored on return */
    if (!on_device.ok) return (int)cudaErrorInvalidDevice;
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    const uint32_t iters = 4096;
    uint32_t *dT0 = nullptr, *sink = nullptr;
    unsigned long long *cyc = nullptr;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    bool ok = cudaMalloc(&dT0, 1024) == cudaSuccess && cudaMalloc(&sink, 16) == cudaSuccess &&
              cudaMalloc(&cyc, sizeof(unsigned long long) * 2 * sms) == cudaSuccess;
    ok = ok && cudaMemcpy(dT0, aesoff_T0_table(), 1024, cudaMemcpyHostToDevice) == cudaSuccess;
    const size_t smem = 196608;
    ok = ok && cudaFuncSetAttribute(calib_lookup_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess;
    double res[3] = {0, 0, 0}, mhz = 0;
    for (int mode = 0; ok && mode < 3; ++mode) {
        const int with_loads = mode == 0 ? 1 : mode == 1 ? 0 : mode;
        calib_lookup_kernel<<<sms, CALIB_THREADS, smem>>>(dT0, 64, sink, cyc, with_loads); /* warm-up */
        cudaEventRecord(e0);
        calib_lookup_kernel<<<sms, CALIB_THREADS, smem>>>(dT0, iters, sink, cyc, with_loads);
        cudaEventRecord(e1);
        ok = cudaEventSynchronize(e1) == cudaSuccess;
        unsigned long long c0 = 0, ns0 = 0;
        ok = ok && cudaMemcpy(&c0, cyc, sizeof(c0), cudaMemcpyDeviceToHost) == cudaSuccess;
        ok = ok && cudaMemcpy(&ns0, cyc + sms, sizeof(ns0), cudaMemcpyDeviceToHost) == cudaSuccess;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        /* per CTA: 16 warps x iters x 16 lookups (warp-wide) in c0 cycles */
        const double ops = (double)(CALIB_THREADS / 32) * iters * CALIB_CHAINS;
        /* alu: 4 PRMT + 4 LOP3 per 4 chains; round: 16 lookups per 4 chains */
        res[mode] = with_loads == 1 ? ops / (double)c0 : with_loads == 0 ? ops * 2.0 / (double)c0 : ops * 4.0 / (double)c0;
        /* in-kernel cycles over in-kernel globaltimer nanoseconds (an event time would include launch and table fill) */
        if (with_loads == 1 && ns0) mhz = (double)c0 * 1e3 / (double)ns0;
    }
    /* bitsliced S-box: verified, then timed */
    double bs_rate = 0, bs_bad = -1;
    {
        uint32_t *mm = nullptr;
        if (ok && cudaMalloc(&mm, 4) == cudaSuccess) {
            const uint32_t bs_iters = 2048;
            cudaMemset(mm, 0, 4);
            calib_bitslice_kernel<<<sms, CALIB_THREADS>>>(dT0, 16, sink, cyc, mm);
            calib_bitslice_kernel<<<sms, CALIB_THREADS>>>(dT0, bs_iters, sink, cyc, mm);
            unsigned long long c0 = 0;
            uint32_t bad = 0;
            ok = cudaDeviceSynchronize() == cudaSuccess && cudaMemcpy(&c0, cyc, sizeof(c0), cudaMemcpyDeviceToHost) == cudaSuccess &&
                 cudaMemcpy(&bad, mm, 4, cudaMemcpyDeviceToHost) == cudaSuccess;
            if (ok && c0) bs_rate = (double)(CALIB_THREADS / 32) * bs_iters * BS_CHAINS / (double)c0;
            bs_bad = (double)bad;
            cudaFree(mm);
        }
    }
    /* copy: 2 x 1 GiB, three passes, best */
    double copy_gbs = 0;
    uint4 *a = nullptr, *b = nullptr;
    const size_t bytes = (size_t)1 << 30;
    if (ok && cudaMalloc(&a, bytes) == cudaSuccess && cudaMalloc(&b, bytes) == cudaSuccess) {
        cudaMemset(a, 1, bytes);
        for (int rep = 0; rep < 4; ++rep) {
            cudaEventRecord(e0);
            calib_copy_kernel<<<sms * 8, CALIB_THREADS>>>(a, b, bytes / 16);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
            float ms = 0;
            cudaEventElapsedTime(&ms, e0, e1);
            const double g = 2.0 * (double)bytes / (ms * 1e-3) / 1e9;
            if (rep > 0 && g > copy_gbs) copy_gbs = g;
        }
    }
    if (a) cudaFree(a);
    if (b) cudaFree(b);
    if (dT0) cudaFree(dT0);
    if (sink) cudaFree(sink);
    if (cyc) cudaFree(cyc);
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (!ok) {
        cudaGetLastError();
        return -1;
    }
    out[0] = res[0];
    out[1] = res[1];
    out[2] = copy_gbs;
    out[3] = mhz;
    out[4] = (double)sms;
    out[5] = res[2];
    out[6] = bs_rate;
    out[7] = bs_bad;
    return 0;
}
