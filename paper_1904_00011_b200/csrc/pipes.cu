// pipes.cu -- instruction-pipe micro-benchmarks behind pcmd_pipe_bench (include/pcmd.h).  They
// measure, on the device the library runs on, the sustained issue rate of the instruction streams the
// stage-2 roofline argument of DESIGN.md "Rooflines" rests on (wide integer multiply of the Philox
// rounds, three-input logic, compare + predicated add, FP32 FMA, shared-memory broadcast / gather)
// and the rate of a kernel that does nothing but Philox4x32-10 (the ceiling of any stage-2 kernel that
// follows R-C1).  `bench.py --pipes` prints the table; nothing on the hot path depends on this file.
#include "pcmd_internal.cuh"

#define PB_CHAINS 8

enum {
    PB_IMAD_WIDE = 0,   // mul.wide.u32 chains (high word | 1 fed back: adds one LOP3 per step, counted)
    PB_LOP3,            // three-input xor chains
    PB_PHILOX_ROUND,    // mul.wide.u32 + lop3 per step (the Philox round pattern)
    PB_FFMA,            // fma.rn.f32, three register operands
    PB_FFMA2,           // fma.rn.f32x2 (two FMAs per instruction)
    PB_SETP_FADD,       // setp.gt.u32 + predicated add.f32 (count a threshold)
    PB_SETP_IADD,       // setp.gt.u32 + predicated add.u32
    PB_PHILOX,          // full Philox4x32-10 calls, counter incremented per call
    PB_LDS_BCAST,       // ld.shared.u32, one address per warp
    PB_LDS_GATHER,      // ld.shared.u32, 32 distinct banks per warp, address-dependent chain
    PB_FADD2,           // add.rn.f32x2
    PB_ROUND_CMP1,      // Philox round step + 1 x (setp + predicated add.f32) on an independent chain
    PB_ROUND_CMP2,      // Philox round step + 2 x (setp + predicated add.f32)
    PB_ROUND_FFMA2,     // Philox round step + 2 x fma.rn.f32
    PB_LOP3_FFMA,       // xor3 + fma.rn.f32 on independent chains
    PB_LOP3_SETP,       // xor3 + setp (+ predicated add.f32) on independent chains
    PB_WIDE_FFMA,       // mul.wide.u32 (hi fed back) + fma.rn.f32
    PB_WIDE_HI,         // mul.wide.u32, high word fed back through prmt-free move (hi ^ lo by one lop3, counted)
    PB_FADD_IMM,        // add.f32 with an immediate
    PB_FFMA_RRR,        // fma.rn.f32 with three varying register operands
    PB_WIDE_FADD,       // mul.wide.u32 + lop3 + add.f32 imm
    PB_WIDE_2FADD,      // mul.wide.u32 + lop3 + 2 x add.f32 imm
    PB_LOP3_IADD,       // xor3 + add.u32 imm on independent chains
    PB_WIDE_IADD,       // mul.wide.u32 + lop3 + 2 x add.u32 imm
    PB_WIDE_FFMA_RRR,   // mul.wide.u32 + lop3 + 2 x fma.rn.f32 (three registers)
    PB_ROUND_CARRY2,    // Philox round + 2 x (add.cc + addc): count a threshold with the integer adder's carry
    PB_ROUND_PIADD2,    // Philox round + 2 x (setp + predicated add.u32)
    PB_ROUND_SELP2,     // Philox round + 2 x (setp + selp.f32 + add.f32)
    PB_ROUND_FFMA2X,    // Philox round + 1 x fma.rn.f32x2
    PB_ROUND_LDS2,      // Philox round + 2 x ld.shared gather
    PB_CARRY,           // add.cc + addc alone
    PB_N
};

static const char *const pb_names[PB_N] = {
    "IMAD.WIDE.U32 (mul.wide.u32)", "LOP3 (xor3)", "IMAD.WIDE.U32 + LOP3 (Philox round)",
    "FFMA (3 registers)", "FFMA2 (fma.rn.f32x2)", "ISETP + predicated FADD", "ISETP + predicated IADD",
    "Philox4x32-10 call", "LDS.32 broadcast", "LDS.32 gather (conflict-free)", "FADD2 (add.rn.f32x2)",
    "Philox round + 1 x (ISETP + pred. FADD)", "Philox round + 2 x (ISETP + pred. FADD)", "Philox round + 2 x FFMA",
    "LOP3 + FFMA", "LOP3 + ISETP + pred. FADD", "IMAD.WIDE.U32 + LOP3(or) + FFMA", "IMAD.WIDE.U32 + LOP3(xor2)",
    "FADD (imm)", "FFMA (R,R,R)", "Philox round + FADD (imm)", "Philox round + 2 x FADD (imm)", "LOP3 + IADD (imm)",
    "Philox round + 2 x IADD (imm)", "Philox round + 2 x FFMA (R,R,R)",
    "Philox round + 2 x (IADD3.CC + IADD3.X)", "Philox round + 2 x (ISETP + pred. IADD)", "Philox round + 2 x (ISETP + FSEL + FADD)",
    "Philox round + FFMA2", "Philox round + 2 x LDS gather", "IADD3.CC + IADD3.X"};
// instructions of interest per chain step (what `rate` counts)
static const int pb_instr[PB_N] = {2, 1, 2, 1, 1, 2, 2, 1, 1, 1, 1, 4, 6, 4, 2, 3, 3, 2, 1, 1, 3, 4, 2, 4, 4, 6, 6, 8, 3, 4, 2};

template <int TEST>
__global__ void k_pipe(int iters, uint32_t a0, uint32_t a1, float f0, float f1, long long *cycles, uint32_t *sink) {
    __shared__ uint32_t tab[64];
    if (threadIdx.x < 64) tab[threadIdx.x] = (threadIdx.x * 17u + 5u) & 31u;
    __syncthreads();
    uint32_t x[PB_CHAINS];
    unsigned long long w[PB_CHAINS];
    float f[PB_CHAINS], g[PB_CHAINS], h[PB_CHAINS];
    uint32_t w32[PB_CHAINS], v32[PB_CHAINS];
#pragma unroll
    for (int k = 0; k < PB_CHAINS; ++k) {
        x[k] = threadIdx.x * 2654435761u + k * 40503u + a0;
        w[k] = x[k];
        f[k] = (float)(x[k] & 1023u) * 1e-3f;
        g[k] = f[k] + 1.0f;
        h[k] = f[k] + 2.0f;
        w32[k] = x[k] >> 3; v32[k] = x[k] >> 5;
    }
    const long long t0 = clock64();
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int rep = 0; rep < 4; ++rep) {
#pragma unroll
            for (int k = 0; k < PB_CHAINS; ++k) {
                if (TEST == PB_IMAD_WIDE) {
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[k]) : "r"((uint32_t)(w[k] >> 32) | 1u), "r"(0xD2511F53u));
                } else if (TEST == PB_LOP3) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[k]) : "r"(a0), "r"(a1));
                } else if (TEST == PB_PHILOX_ROUND) {
                    unsigned long long p;
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x[k]), "r"(0xD2511F53u));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[k]) : "r"((uint32_t)p), "r"((uint32_t)(p >> 32)), "r"(a1));
                } else if (TEST == PB_ROUND_CMP1 || TEST == PB_ROUND_CMP2 || TEST == PB_ROUND_FFMA2) {
                    unsigned long long p;
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x[k]), "r"(0xD2511F53u));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[k]) : "r"((uint32_t)p), "r"((uint32_t)(p >> 32)), "r"(a1));
                    if (TEST == PB_ROUND_FFMA2) {
                        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[k]) : "f"(f0), "f"(f1));
                        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(g[k]) : "f"(f0), "f"(f1));
                    } else {
                        asm volatile("{\n.reg .pred p;\nsetp.gt.u32 p, %1, %2;\n@p add.f32 %0, %0, 0f3F800000;\n}"
                                     : "+f"(f[k]) : "r"(__float_as_uint(f[k])), "r"(a1));
                        if (TEST == PB_ROUND_CMP2)
                            asm volatile("{\n.reg .pred p;\nsetp.gt.u32 p, %1, %2;\n@p add.f32 %0, %0, 0f3F800000;\n}"
                                         : "+f"(g[k]) : "r"(__float_as_uint(g[k])), "r"(a1));
                    }
                } else if (TEST == PB_LOP3_FFMA) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[k]) : "r"(a0), "r"(a1));
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[k]) : "f"(f0), "f"(f1));
                } else if (TEST == PB_LOP3_SETP) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[k]) : "r"(a0), "r"(a1));
                    asm volatile("{\n.reg .pred p;\nsetp.gt.u32 p, %1, %2;\n@p add.f32 %0, %0, 0f3F800000;\n}"
                                 : "+f"(f[k]) : "r"(__float_as_uint(f[k])), "r"(a1));
                } else if (TEST == PB_WIDE_FFMA) {
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[k]) : "r"((uint32_t)(w[k] >> 32) | 1u), "r"(0xD2511F53u));
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[k]) : "f"(f0), "f"(f1));
                } else if (TEST == PB_WIDE_HI) {
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(w[k]) : "r"((uint32_t)(w[k] >> 32) ^ (uint32_t)w[k]), "r"(0xD2511F53u));
                } else if (TEST == PB_FADD_IMM) {
                    asm volatile("add.f32 %0, %0, 0f3F800000;" : "+f"(f[k]));
                } else if (TEST == PB_FFMA_RRR) {
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[k]) : "f"(g[k]), "f"(g[(k + 1) & 7]));
                } else if (TEST == PB_WIDE_FADD || TEST == PB_WIDE_2FADD || TEST == PB_WIDE_IADD || TEST == PB_WIDE_FFMA_RRR) {
                    unsigned long long p;
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x[k]), "r"(0xD2511F53u));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[k]) : "r"((uint32_t)p), "r"((uint32_t)(p >> 32)), "r"(a1));
                    if (TEST == PB_WIDE_IADD) {
                        asm volatile("add.u32 %0, %0, 3;" : "+r"(w32[k]));
                        asm volatile("add.u32 %0, %0, 5;" : "+r"(v32[k]));
                    } else if (TEST == PB_WIDE_FFMA_RRR) {
                        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[k]) : "f"(g[k]), "f"(g[(k + 1) & 7]));
                        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(h[k]) : "f"(g[k]), "f"(g[(k + 2) & 7]));
                    } else {
                        asm volatile("add.f32 %0, %0, 0f3F800000;" : "+f"(f[k]));
                        if (TEST == PB_WIDE_2FADD) asm volatile("add.f32 %0, %0, 0f3F800000;" : "+f"(g[k]));
                    }
                } else if (TEST == PB_ROUND_CARRY2 || TEST == PB_ROUND_PIADD2 || TEST == PB_ROUND_SELP2 || TEST == PB_ROUND_FFMA2X || TEST == PB_ROUND_LDS2) {
                    unsigned long long p;
                    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x[k]), "r"(0xD2511F53u));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[k]) : "r"((uint32_t)p), "r"((uint32_t)(p >> 32)), "r"(a1));
                    if (TEST == PB_ROUND_CARRY2) {
                        asm volatile("{\n.reg .u32 t;\nadd.cc.u32 t, %0, %1;\naddc.u32 %0, %0, 0;\n}" : "+r"(w32[k]) : "r"(a1));
                        asm volatile("{\n.reg .u32 t;\nadd.cc.u32 t, %0, %1;\naddc.u32 %0, %0, 0;\n}" : "+r"(v32[k]) : "r"(a0));
                    } else if (TEST == PB_ROUND_PIADD2) {
                        asm volatile("{\n.reg .pred q;\nsetp.gt.u32 q, %0, %1;\n@q add.u32 %0, %0, 1;\n}" : "+r"(w32[k]) : "r"(a1));
                        asm volatile("{\n.reg .pred q;\nsetp.gt.u32 q, %0, %1;\n@q add.u32 %0, %0, 1;\n}" : "+r"(v32[k]) : "r"(a0));
                    } else if (TEST == PB_ROUND_SELP2) {
                        asm volatile("{\n.reg .pred q;\n.reg .f32 t;\nsetp.gt.u32 q, %1, %2;\nselp.f32 t, 0f3F800000, 0f00000000, q;\nadd.f32 %0, %0, t;\n}"
                                     : "+f"(f[k]) : "r"(__float_as_uint(f[k])), "r"(a1));
                        asm volatile("{\n.reg .pred q;\n.reg .f32 t;\nsetp.gt.u32 q, %1, %2;\nselp.f32 t, 0f3F800000, 0f00000000, q;\nadd.f32 %0, %0, t;\n}"
                                     : "+f"(g[k]) : "r"(__float_as_uint(g[k])), "r"(a1));
                    } else if (TEST == PB_ROUND_FFMA2X) {
                        unsigned long long acc, m, c;
                        asm volatile("mov.b64 %0, {%1, %2};" : "=l"(acc) : "f"(f[k]), "f"(g[k]));
                        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(f0));
                        asm volatile("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(f1));
                        asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(acc) : "l"(m), "l"(c));
                        asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(f[k]), "=f"(g[k]) : "l"(acc));
                    } else {
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(w32[k]) : "r"((uint32_t)__cvta_generic_to_shared(tab) + 4u * ((w32[k] + threadIdx.x) & 31u)));
                        asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v32[k]) : "r"((uint32_t)__cvta_generic_to_shared(tab) + 4u * ((v32[k] + threadIdx.x) & 31u)));
                    }
                } else if (TEST == PB_CARRY) {
                    asm volatile("{\n.reg .u32 t;\nadd.cc.u32 t, %0, %1;\naddc.u32 %0, %0, 0;\n}" : "+r"(w32[k]) : "r"(a1));
                } else if (TEST == PB_LOP3_IADD) {
                    asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[k]) : "r"(a0), "r"(a1));
                    asm volatile("add.u32 %0, %0, 3;" : "+r"(w32[k]));
                } else if (TEST == PB_FFMA) {
                    asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(f[k]) : "f"(f0), "f"(f1));
                } else if (TEST == PB_FFMA2) {
                    unsigned long long acc, m, c;
                    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(acc) : "f"(f[k]), "f"(g[k]));
                    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(m) : "f"(f0));
                    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(f1));
                    asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(acc) : "l"(m), "l"(c));
                    asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(f[k]), "=f"(g[k]) : "l"(acc));
                } else if (TEST == PB_FADD2) {
                    unsigned long long acc, c;
                    asm volatile("mov.b64 %0, {%1, %2};" : "=l"(acc) : "f"(f[k]), "f"(g[k]));
                    asm volatile("mov.b64 %0, {%1, %1};" : "=l"(c) : "f"(f1));
                    asm volatile("add.rn.f32x2 %0, %0, %1;" : "+l"(acc) : "l"(c));
                    asm volatile("mov.b64 {%0, %1}, %2;" : "=f"(f[k]), "=f"(g[k]) : "l"(acc));
                } else if (TEST == PB_SETP_FADD) {
                    asm volatile("{\n.reg .pred p;\nsetp.gt.u32 p, %1, %2;\n@p add.f32 %0, %0, 0f3F800000;\n}"
                                 : "+f"(f[k]) : "r"(__float_as_uint(f[k])), "r"(a1));
                } else if (TEST == PB_SETP_IADD) {
                    asm volatile("{\n.reg .pred p;\nsetp.gt.u32 p, %0, %1;\n@p add.u32 %0, %0, 1;\n}"
                                 : "+r"(x[k]) : "r"(a1));
                } else if (TEST == PB_PHILOX) {
                    if (k < 2 && rep < 2) {      // 4 calls per iteration, two independent at a time
                        uint32_t o[4];
                        philox4x32_10(a0, a1, x[k], (uint32_t)it, 7u, 0u, o);
                        x[k] += o[0] ^ o[1] ^ o[2] ^ o[3];
                    }
                } else if (TEST == PB_LDS_BCAST) {
                    uint32_t v;
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"((uint32_t)__cvta_generic_to_shared(tab) + 4u * ((it + k + 8 * rep) & 63)));
                    x[k] ^= v;
                } else if (TEST == PB_LDS_GATHER) {
                    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(x[k]) : "r"((uint32_t)__cvta_generic_to_shared(tab) + 4u * ((x[k] + threadIdx.x) & 31u)));
                }
            }
        }
    }
    const long long t1 = clock64();
    uint32_t s = 0;
#pragma unroll
    for (int k = 0; k < PB_CHAINS; ++k) s ^= x[k] ^ (uint32_t)w[k] ^ (uint32_t)(w[k] >> 32) ^ __float_as_uint(f[k]) ^ __float_as_uint(g[k]) ^ __float_as_uint(h[k]) ^ w32[k] ^ v32[k];
    if (s == 0x12345678u) sink[0] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

template <int TEST>
static cudaError_t pb_launch(int grid, int threads, int iters, long long *d_cyc, uint32_t *d_sink) {
    k_pipe<TEST><<<grid, threads>>>(iters, 0x9E3779B9u, 0x7F4A7C15u, 0.999f, 1e-3f, d_cyc, d_sink);
    return cudaGetLastError();
}

extern "C" const char *pcmd_pipe_bench_name(int32_t test) {
    return (test >= 0 && test < PB_N) ? pb_names[test] : nullptr;
}

extern "C" int pcmd_pipe_bench(int32_t test, int32_t ctas_per_sm, int32_t threads, int32_t iters, double *h_out) {
    if (test < 0 || test >= PB_N || ctas_per_sm < 1 || threads < 32 || threads > 1024 || (threads & 31) || iters < 1 || !h_out)
        return PCMD_EINVAL;
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const int grid = sms * ctas_per_sm;
    long long *d_cyc = nullptr; uint32_t *d_sink = nullptr;
    if (cudaMalloc(&d_cyc, grid * sizeof(long long)) != cudaSuccess) return PCMD_ENOMEM;
    if (cudaMalloc(&d_sink, 16) != cudaSuccess) { cudaFree(d_cyc); return PCMD_ENOMEM; }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaError_t e = cudaSuccess;
    float ms = 0.f;
    for (int pass = 0; pass < 2 && e == cudaSuccess; ++pass) {      // warm-up pass, timed pass
        cudaEventRecord(e0);
        switch (test) {
            case PB_IMAD_WIDE: e = pb_launch<PB_IMAD_WIDE>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_LOP3: e = pb_launch<PB_LOP3>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_PHILOX_ROUND: e = pb_launch<PB_PHILOX_ROUND>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_FFMA: e = pb_launch<PB_FFMA>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_FFMA2: e = pb_launch<PB_FFMA2>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_SETP_FADD: e = pb_launch<PB_SETP_FADD>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_SETP_IADD: e = pb_launch<PB_SETP_IADD>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_PHILOX: e = pb_launch<PB_PHILOX>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_LDS_BCAST: e = pb_launch<PB_LDS_BCAST>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_LDS_GATHER: e = pb_launch<PB_LDS_GATHER>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_FADD2: e = pb_launch<PB_FADD2>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_CMP1: e = pb_launch<PB_ROUND_CMP1>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_CMP2: e = pb_launch<PB_ROUND_CMP2>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_FFMA2: e = pb_launch<PB_ROUND_FFMA2>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_LOP3_FFMA: e = pb_launch<PB_LOP3_FFMA>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_LOP3_SETP: e = pb_launch<PB_LOP3_SETP>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_WIDE_FFMA: e = pb_launch<PB_WIDE_FFMA>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_WIDE_HI: e = pb_launch<PB_WIDE_HI>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_FADD_IMM: e = pb_launch<PB_FADD_IMM>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_FFMA_RRR: e = pb_launch<PB_FFMA_RRR>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_WIDE_FADD: e = pb_launch<PB_WIDE_FADD>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_WIDE_2FADD: e = pb_launch<PB_WIDE_2FADD>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_LOP3_IADD: e = pb_launch<PB_LOP3_IADD>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_WIDE_IADD: e = pb_launch<PB_WIDE_IADD>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_WIDE_FFMA_RRR: e = pb_launch<PB_WIDE_FFMA_RRR>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_CARRY2: e = pb_launch<PB_ROUND_CARRY2>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_PIADD2: e = pb_launch<PB_ROUND_PIADD2>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_SELP2: e = pb_launch<PB_ROUND_SELP2>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_FFMA2X: e = pb_launch<PB_ROUND_FFMA2X>(grid, threads, iters, d_cyc, d_sink); break;
            case PB_ROUND_LDS2: e = pb_launch<PB_ROUND_LDS2>(grid, threads, iters, d_cyc, d_sink); break;
            default: e = pb_launch<PB_CARRY>(grid, threads, iters, d_cyc, d_sink); break;
        }
        cudaEventRecord(e1);
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    }
    double cyc_max = 0.0;
    if (e == cudaSuccess) {
        cudaEventElapsedTime(&ms, e0, e1);
        long long *h = (long long *)malloc(grid * sizeof(long long));
        if (h) {
            e = cudaMemcpy(h, d_cyc, grid * sizeof(long long), cudaMemcpyDeviceToHost);
            for (int i = 0; i < grid; ++i) if ((double)h[i] > cyc_max) cyc_max = (double)h[i];
            free(h);
        }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(d_cyc); cudaFree(d_sink);
    if (e != cudaSuccess) return PCMD_ECUDA;
    // steps per thread: iters x 4 x PB_CHAINS (Philox: 4 calls per iteration)
    const double steps = test == PB_PHILOX ? (double)iters * 4.0 : (double)iters * 4.0 * PB_CHAINS;
    const double warps_per_sched = (double)ctas_per_sm * (threads / 32) / 4.0;
    h_out[0] = steps * pb_instr[test] * warps_per_sched / cyc_max;     // warp-instructions (or calls) / clk / scheduler
    h_out[1] = cyc_max;
    h_out[2] = (double)ms;
    h_out[3] = steps * (double)grid * threads / ((double)ms * 1e-3);   // thread-steps per second over the GPU
    return PCMD_OK;
}
