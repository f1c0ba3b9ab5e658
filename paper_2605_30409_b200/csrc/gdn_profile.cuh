// gdn_profile.cuh -- optional per-kernel CUDA-event timing (gdn_plan_set_profiling / gdn_plan_kernel_times).
#pragma once
#include <cuda_runtime.h>

#include <vector>

namespace gdn {

class Profiler {
  public:
    void set_enabled(bool on) {
        if (!on) clear();
        enabled_ = on;
    }
    bool enabled() const { return enabled_; }
    // before the first kernel of a call
    void begin(cudaStream_t st) {
        if (!enabled_) return;
        calls_.emplace_back();
        push(st, nullptr);
    }
    // after each kernel of the call
    void mark(cudaStream_t st, const char* name) {
        if (!enabled_ || calls_.empty()) return;
        push(st, name);
    }
    // -> number of kernels; averages over the recorded calls; clears the events
    int collect(int max_n, const char** names, float* avg_ms) {
        int n = 0;
        std::vector<double> sum;
        std::vector<const char*> nm;
        for (auto& call : calls_) {
            for (size_t i = 1; i < call.size(); ++i) {
                cudaEventSynchronize(call[i].ev);
                float ms = 0.f;
                cudaEventElapsedTime(&ms, call[i - 1].ev, call[i].ev);
                if (sum.size() < i) { sum.push_back(0.0); nm.push_back(call[i].name); }
                sum[i - 1] += ms;
            }
        }
        const double nc = calls_.empty() ? 1.0 : (double)calls_.size();
        for (size_t i = 0; i < sum.size() && n < max_n; ++i, ++n) { names[n] = nm[i]; avg_ms[n] = (float)(sum[i] / nc); }
        clear();
        return n;
    }

  private:
    struct Mark { cudaEvent_t ev; const char* name; };
    void push(cudaStream_t st, const char* name) {
        Mark m{nullptr, name};
        cudaEventCreate(&m.ev);
        cudaEventRecord(m.ev, st);
        calls_.back().push_back(m);
    }
    void clear() {
        for (auto& call : calls_) for (auto& m : call) cudaEventDestroy(m.ev);
        calls_.clear();
    }
    bool enabled_ = false;
    std::vector<std::vector<Mark>> calls_;
};

}  // namespace gdn
