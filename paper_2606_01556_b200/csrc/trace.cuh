// trace.cuh -- optional in-kernel timeline, compiled in ONLY by `python -m paper_2606_01556_b200._build --trace`
// (-DTWQ_TRACE, library libtwq_trace.so).  The product library contains none of it: the macros below are empty.
//
// The caller hands a device buffer to the library with twq_testing_set_trace_buffer (include/twq_testing.h); the
// launchers copy the pointer into the kernel parameters.
//   decode kernel : TWQ_DSTAMP(k) -- lane 0 of every warp of CTA 0 and of CTA grid/2 stores %globaltimer (ns) at
//                   buffer[((cta_sel * 20 + warp) * 64) + k], k < 32;
//                   TWQ_DCLK(k) stores clock64 (SM cycles) at slot 32 + k of the same row.
//   tcgen05 kernel: TWQ_TR(role, n, tag) -- CTA 0 appends (tag << 48 | clock64) to buffer[role * 4096 + n++], four roles;
//                   TWQ_TG(k) -- whole-kernel milestones (clock64) of CTA 0 at buffer[4 * 4096 - 64 + k].
#pragma once

#ifdef TWQ_TRACE
#define TWQ_DSTAMP(k)                                                                                    \
    do {                                                                                                 \
        if (p.trace != nullptr && (threadIdx.x & 31) == 0 && (blockIdx.x == 0 || blockIdx.x == gridDim.x / 2)) { \
            unsigned long long t_;                                                                       \
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t_));                                       \
            p.trace[(((blockIdx.x != 0) * 20 + (threadIdx.x >> 5)) * 64) + (k)] = t_;                     \
        }                                                                                                \
    } while (0)
/* fine-grained: SM cycle counter into slots 32..63 of the same row (cheap: no timer read, one store) */
#define TWQ_DCLK(k)                                                                                      \
    do {                                                                                                 \
        if (p.trace != nullptr && (threadIdx.x & 31) == 0 && (blockIdx.x == 0 || blockIdx.x == gridDim.x / 2)) \
            p.trace[(((blockIdx.x != 0) * 20 + (threadIdx.x >> 5)) * 64) + 32 + (k)] =                    \
                static_cast<unsigned long long>(clock64());                                              \
    } while (0)
#define TWQ_TR(role, n, tag)                                                                             \
    do {                                                                                                 \
        if (p.trace != nullptr && blockIdx.x == 0 && (n) < 4096)                                         \
            p.trace[(role) * 4096 + (n)++] = (static_cast<unsigned long long>(tag) << 48) |              \
                                             (static_cast<unsigned long long>(clock64()) & 0xFFFFFFFFFFFFull); \
    } while (0)
/* tcgen05 kernel, whole-kernel milestones: thread 256 (first epilogue thread) of CTA 0 stores clock64 at buffer[4 * 4096 - 64 + k] */
#define TWQ_TG(k)                                                                                        \
    do {                                                                                                 \
        if (p.trace != nullptr && blockIdx.x == 0 && threadIdx.x == 256)                                 \
            p.trace[4 * 4096 - 64 + (k)] = static_cast<unsigned long long>(clock64());                   \
    } while (0)
#else
#define TWQ_TG(k) do { } while (0)
#define TWQ_DSTAMP(k) do { } while (0)
#define TWQ_DCLK(k) do { } while (0)
#define TWQ_TR(role, n, tag) do { } while (0)
#endif
