// sc_probe.h -- optional in-kernel timeline of the tcgen05 attention kernel.
// Compiled out unless the library is built with -DSC_TC_PROBE (a development build; the product
// build never defines it).  TL(i) stores clock64() of one thread of the CTA into slot i of a
// per-CTA record, TLG(i) the global timer; PROBE(bit) tests a run-time flag that switches a
// phase of the kernel off (results are then wrong: timing experiments only).
#pragma once

#ifdef SC_TC_PROBE
__constant__ int sc_probe_flags;
__device__ long long sc_tl[256][64];
__device__ long long sc_lt[256][2];          // per launch (mod 256): global timer at start / end of CTA 0
__device__ unsigned int sc_launch_no;
#define PROBE(bit) (sc_probe_flags & (1 << (bit)))
#define TL(i) do { const int cta_ = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z); \
                   if (cta_ < 256) sc_tl[cta_][(i)] = clock64(); } while (0)
#define TLG(i) do { const int cta_ = blockIdx.x + gridDim.x * (blockIdx.y + gridDim.y * blockIdx.z); \
                    long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); \
                    if (cta_ < 256) sc_tl[cta_][(i)] = t_; } while (0)
#define LAUNCH_BEGIN() do { if (blockIdx.x + blockIdx.y + blockIdx.z == 0 && threadIdx.x == 0) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); sc_lt[sc_launch_no & 255][0] = t_; } } while (0)
#define LAUNCH_END() do { if (blockIdx.x + blockIdx.y + blockIdx.z == 0 && threadIdx.x == 128) { long long t_; asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_)); sc_lt[sc_launch_no & 255][1] = t_; sc_launch_no += 1; } } while (0)
#else
#define LAUNCH_BEGIN() do { } while (0)
#define LAUNCH_END() do { } while (0)
#define PROBE(bit) 0
#define TL(i) do { } while (0)
#define TLG(i) do { } while (0)
#endif
