// mr_stream.cuh -- streaming TMA step kernel (placeholder until the kernel lands; the generic path is used).
#pragma once
#include <string>
#include "mr_common.cuh"

namespace mr {

struct StreamGeom {
    int nx, ny, nz, pitch;
    long long plane, comp;
    double twoh[3];
};

struct StreamPlan {
    bool usable = false;
    const char* name = "stream";
    std::string why;
};

inline bool build_stream_plan(StreamPlan* p, const StreamGeom&, bool, void*, void*, void*, int, std::string* why)
{
    p->usable = false;
    *why = "streaming kernel not built";
    return false;
}

template <typename T>
inline cudaError_t launch_stream_step(const StreamPlan&, int, T, int*, cudaStream_t)
{
    return cudaErrorNotSupported;
}

}  // namespace mr
