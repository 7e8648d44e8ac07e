// Developer instrumentation for the tcgen05 kernels, compiled out unless the library is built with -DWM_TC_PROFILE
// (WM_TC_PROFILE=1 python -m paper_2606_09312_b200.build --force) AND the process sets WM_TC_PROF=<file>: lane 0 of one
// warp per role of CTA 0 appends (tag, clock) records to a device buffer that the launcher dumps as "role tag clock"
// lines.  Nothing of this exists in a normal build: the macros expand to nothing and Params::prof stays null.
#pragma once

#include <cstdio>
#include <cstdlib>
#include <vector>

#include "wm_internal.h"

namespace wm {
namespace trace {

constexpr int CAP = 16384;     // records per role
constexpr int ROLES = 4;       // 0 = MMA issuer, 1 = producer, 2 = epilogue warp 0, 3 = action warp 0

#ifdef WM_TC_PROFILE
#define WM_TRACE_DECL(prof, role)                                                                                  \
    uint2* tr_buf = (prof) ? reinterpret_cast<uint2*>(prof) + (role) * ::wm::trace::CAP : nullptr;                 \
    const bool tr_on = tr_buf != nullptr && blockIdx.x == 0 && lane == 0;                                          \
    uint32_t tr_n = 0;
#define WM_TRACE(tag)                                                                                              \
    do {                                                                                                           \
        if (tr_on && tr_n < ::wm::trace::CAP - 1) {                                                                \
            tr_buf[1 + tr_n] = make_uint2((uint32_t)(tag), (uint32_t)clock64());                                   \
            ++tr_n;                                                                                                \
            tr_buf[0].x = tr_n;                                                                                    \
        }                                                                                                          \
    } while (0)

// host: a zeroed trace buffer when WM_TC_PROF is set, else nullptr
inline unsigned long long* begin(cudaStream_t st) {
    static unsigned long long* d_prof = nullptr;
    if (!getenv("WM_TC_PROF")) return nullptr;
    const size_t bytes = (size_t)ROLES * CAP * 8;
    if (!d_prof && cudaMalloc(&d_prof, bytes) != cudaSuccess) return nullptr;
    cudaMemsetAsync(d_prof, 0, bytes, st);
    return d_prof;
}
// host: wait for the launch and write the records to WM_TC_PROF's path
inline void dump(unsigned long long* prof, cudaStream_t st) {
    if (!prof) return;
    std::vector<uint2> h((size_t)ROLES * CAP);
    cudaStreamSynchronize(st);
    cudaMemcpy(h.data(), prof, h.size() * 8, cudaMemcpyDeviceToHost);
    FILE* f = fopen(getenv("WM_TC_PROF"), "w");
    if (!f) return;
    for (int r = 0; r < ROLES; ++r)
        for (uint32_t i = 0; i < h[(size_t)r * CAP].x; ++i)
            fprintf(f, "%d %u %u\n", r, h[(size_t)r * CAP + 1 + i].x, h[(size_t)r * CAP + 1 + i].y);
    fclose(f);
}
#else
#define WM_TRACE_DECL(prof, role)
#define WM_TRACE(tag) do { } while (0)
inline unsigned long long* begin(cudaStream_t) { return nullptr; }
inline void dump(unsigned long long*, cudaStream_t) {}
#endif

}  // namespace trace
}  // namespace wm
