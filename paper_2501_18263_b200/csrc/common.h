// Shared host-side declarations of the DMRG library (not part of the public C ABI).
#pragma once
#include <cuda_runtime.h>

#include <chrono>
#include <cstdint>
#include <cstdlib>
#include <cstdio>
#include <stdexcept>
#include <string>
#include <unordered_map>
#include <vector>

#include "../../include/dmrg_b200.h"

namespace dmrg {

struct Error : std::runtime_error {
  int code;
  Error(int c, const std::string& m) : std::runtime_error(m), code(c) {}
};

#define DMRG_CUDA(x)                                                                          \
  do {                                                                                        \
    cudaError_t e__ = (x);                                                                    \
    if (e__ != cudaSuccess)                                                                   \
      throw dmrg::Error(DMRG_ERR_CUDA, std::string(#x) + ": " + cudaGetErrorString(e__));     \
  } while (0)

#define DMRG_REQUIRE(cond, code, msg)                 \
  do {                                                \
    if (!(cond)) throw dmrg::Error((code), (msg));    \
  } while (0)

// DMRG_B200_TIMING=1: host-side phase times of the planning code on stderr (measurement aid)
struct PhaseTimer {
  bool on;
  const char* what;
  std::chrono::steady_clock::time_point t;
  explicit PhaseTimer(const char* w) : on(std::getenv("DMRG_B200_TIMING") != nullptr), what(w), t(std::chrono::steady_clock::now()) {}
  void lap(const char* name) {
    if (!on) return;
    auto n = std::chrono::steady_clock::now();
    fprintf(stderr, "[timing] %s: %s %.1f ms\n", what, name, std::chrono::duration<double, std::milli>(n - t).count());
    t = n;
  }
};

inline int pad8(int x) { return (x + 7) & ~7; }

// Device memory through the user's allocator callbacks.
struct Allocator {
  dmrg_alloc_fn alloc = nullptr;
  dmrg_free_fn free_ = nullptr;
  void* user = nullptr;
  uint64_t live_bytes = 0, peak_bytes = 0;
  std::unordered_map<void*, uint64_t> sizes;
  void* get(uint64_t bytes) {
    if (bytes == 0) bytes = 256;
    void* p = alloc(bytes, user);
    if (!p) throw Error(DMRG_ERR_ALLOC, "device allocator returned NULL for " + std::to_string(bytes) + " bytes");
    sizes[p] = bytes;
    live_bytes += bytes;
    if (live_bytes > peak_bytes) peak_bytes = live_bytes;
    return p;
  }
  void put(void* p) {
    if (!p) return;
    auto it = sizes.find(p);
    if (it != sizes.end()) { live_bytes -= it->second; sizes.erase(it); }
    free_(p, user);
  }
};

template <typename T>
struct DevArray {   // owning device array
  Allocator* al = nullptr;
  T* p = nullptr;
  size_t n = 0;
  DevArray() = default;
  DevArray(const DevArray&) = delete;
  DevArray& operator=(const DevArray&) = delete;
  DevArray(DevArray&& o) noexcept { *this = std::move(o); }
  DevArray& operator=(DevArray&& o) noexcept {
    if (this != &o) { release(); al = o.al; p = o.p; n = o.n; o.p = nullptr; o.n = 0; }
    return *this;
  }
  ~DevArray() { release(); }
  void release() { if (p && al) al->put(p); p = nullptr; n = 0; }
  void allocate(Allocator* a, size_t count) {
    release(); al = a; n = count;
    p = static_cast<T*>(a->get(static_cast<uint64_t>(count) * sizeof(T)));
  }
  void upload(Allocator* a, const std::vector<T>& h, cudaStream_t st) {
    allocate(a, h.size());
    if (!h.empty()) DMRG_CUDA(cudaMemcpyAsync(p, h.data(), h.size() * sizeof(T), cudaMemcpyHostToDevice, st));
  }
};

}  // namespace dmrg
