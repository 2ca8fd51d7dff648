// ea_pipes.cu -- ea_selftest_pipes: the measured issue rates that bound the sweep and observable kernels.
//
// The update of the paper is "boolean logic at the bit level" plus one random number (section III):
// on sm_100a that is LOP3 (alu pipe) + IMAD.WIDE.U32 (fma pipe, Philox) for the sweep and POPC for the
// observables (Eq. 3, 7).  SURVEY 8(d) asks for these rates to be MEASURED on the chip ("dependent-free LOP3 and
// IMAD.WIDE streams, all SMs"), because MEASURED_PEAKS.json has no integer figure; bench.py calls this before the
// timed region and reports the sweep kernel against the LOP3 rate measured in the same run.
//
// Every stream is ILP-8 (eight independent accumulators per thread), 32 warps per SM, one CTA per SM on all SMs;
// the instruction count is exact by construction (inline PTX, one instruction per statement; ea_selftest_pipes
// checks nothing else -- tests/test_abi.py counts the opcodes in the SASS of these kernels).
#include "ea_internal.h"

namespace ea {

enum { PIPE_LOP3 = 0, PIPE_IMAD_WIDE = 1, PIPE_POPC = 2, PIPE_MIX = 3, PIPE_MIX_IMAD = 4 };
constexpr int PIPE_ILP = 8, PIPE_UNROLL = 16; // instructions of the measured kind per loop trip: ILP * UNROLL

template <int KIND>
__global__ void __launch_bounds__(1024, 1) k_pipe_stream(uint32_t *out, const int trips, unsigned long long *ticks)
{
    uint32_t a[PIPE_ILP], m[PIPE_ILP];
    uint64_t w[PIPE_ILP];
    const uint32_t b = threadIdx.x * 0x9E3779B9u + 1u, c = blockIdx.x * 0x85EBCA6Bu + 7u;
#pragma unroll
    for (int i = 0; i < PIPE_ILP; ++i) { a[i] = b + i * c; m[i] = a[i] ^ 0x5555u; w[i] = ((uint64_t)a[i] << 32) | (b ^ i); }
    unsigned long long t0 = 0, c0 = 0;
    if (threadIdx.x == 0) {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        c0 = clock64();
    }
#pragma unroll 1
    for (int t = 0; t < trips; ++t) {
#pragma unroll
        for (int u = 0; u < PIPE_UNROLL; ++u) {
#pragma unroll
            for (int i = 0; i < PIPE_ILP; ++i) {
                if (KIND == PIPE_LOP3 || KIND == PIPE_MIX || KIND == PIPE_MIX_IMAD) { // xor3 and maj alternate, so that two never fold into one
                    if (u & 1) asm volatile("lop3.b32 %0, %0, %1, %2, 0xe8;" : "+r"(a[i]) : "r"(a[(i + 1) % PIPE_ILP]), "r"(c));
                    else asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(a[i]) : "r"(a[(i + 1) % PIPE_ILP]), "r"(c));
                }
                // w = hi32(w) * M: the 32 x 32 -> 64 product of a Philox round (the high word feeds the next one, so the
                // chain cannot be folded into one multiply).  The mix issues one per four LOP3, about the sweep kernel's
                // ratio.  MEASURED (B200): the LOP3 rate of the mix is 4/5 of the LOP3 rate alone at every ratio tried --
                // an IMAD.WIDE (or IMAD.HI) takes an issue slot of the alu pipe besides its four clocks on the fma pipe,
                // whereas a plain 32-bit IMAD (the second mix) overlaps with LOP3.  The alu roofline of the sweep kernel
                // therefore counts IMAD.WIDE as alu-pipe work.
                if (KIND == PIPE_IMAD_WIDE || (KIND == PIPE_MIX && i % 4 == 0))
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[i]) : "r"((uint32_t)(w[i] >> 32)), "r"(0xD2511F53u));
                if (KIND == PIPE_MIX_IMAD) // one 32-bit IMAD per LOP3
                    asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(m[i]) : "r"(0xD2511F53u), "r"(c));
                if (KIND == PIPE_POPC)
                    asm volatile("popc.b32 %0, %0;" : "+r"(a[i]));
            }
        }
    }
    if (threadIdx.x == 0) {
        unsigned long long t1, c1 = clock64();
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        ticks[2 * blockIdx.x] = t1 - t0;     // ns
        ticks[2 * blockIdx.x + 1] = c1 - c0; // SM clocks
    }
    uint32_t r = 0;
#pragma unroll
    for (int i = 0; i < PIPE_ILP; ++i) r ^= a[i] ^ m[i] ^ (uint32_t)w[i] ^ (uint32_t)(w[i] >> 32);
    out[blockIdx.x * blockDim.x + threadIdx.x] = r;
}

template <int KIND>
static cudaError_t time_stream(int n_sm, uint32_t *d_out, unsigned long long *d_ticks, int trips, double *rate, double *mhz)
{
    cudaEvent_t e0, e1;
    cudaError_t e = cudaEventCreate(&e0);
    if (e != cudaSuccess) return e;
    if ((e = cudaEventCreate(&e1)) != cudaSuccess) { cudaEventDestroy(e0); return e; }
    float best = 1e30f;
    for (int rep = 0; rep < 4; ++rep) { // first pass warms up; best of the other three
        cudaEventRecord(e0, 0);
        k_pipe_stream<KIND><<<n_sm, 1024>>>(d_out, trips, d_ticks);
        cudaEventRecord(e1, 0);
        if ((e = cudaEventSynchronize(e1)) != cudaSuccess) break;
        float ms = 0;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep && ms < best) best = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (e != cudaSuccess) return e;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    const double warp_inst = (double)n_sm * 32.0 * (double)trips * PIPE_ILP * PIPE_UNROLL;
    *rate = warp_inst / (best * 1e-3);
    if (mhz) { // SM clock during the stream: clock64 ticks / globaltimer ns of CTA 0
        unsigned long long h[2];
        if ((e = cudaMemcpy(h, d_ticks, sizeof(h), cudaMemcpyDeviceToHost)) != cudaSuccess) return e;
        *mhz = h[0] ? 1e3 * (double)h[1] / (double)h[0] : 0.0;
    }
    return cudaSuccess;
}

cudaError_t pipe_rates(int device, double out[8])
{
    int n_sm = 0;
    cudaError_t e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    uint32_t *d_out = nullptr;
    unsigned long long *d_ticks = nullptr;
    if ((e = cudaMalloc(&d_out, (size_t)n_sm * 1024 * sizeof(uint32_t))) != cudaSuccess) return e;
    if ((e = cudaMalloc(&d_ticks, (size_t)n_sm * 2 * sizeof(unsigned long long))) != cudaSuccess) { cudaFree(d_out); return e; }
    const int trips = 4096; // 148 SMs x 32 warps x 4096 x 128 = 2.5 G warp instructions: ~4 ms at the alu rate
    double mhz = 0;
    e = time_stream<PIPE_LOP3>(n_sm, d_out, d_ticks, trips, &out[0], &mhz);
    if (e == cudaSuccess) e = time_stream<PIPE_IMAD_WIDE>(n_sm, d_out, d_ticks, trips, &out[1], nullptr);
    if (e == cudaSuccess) e = time_stream<PIPE_POPC>(n_sm, d_out, d_ticks, trips / 4, &out[2], nullptr);
    if (e == cudaSuccess) e = time_stream<PIPE_MIX>(n_sm, d_out, d_ticks, trips, &out[3], nullptr); // LOP3 count; one IMAD.WIDE per four LOP3 alongside
    out[6] = out[7] = 0.0;
    if (e == cudaSuccess) e = time_stream<PIPE_MIX_IMAD>(n_sm, d_out, d_ticks, trips, &out[6], nullptr); // LOP3 count; as many IMAD
    out[4] = mhz;
    out[5] = (double)n_sm;
    cudaFree(d_out);
    cudaFree(d_ticks);
    return e;
}

} // namespace ea
