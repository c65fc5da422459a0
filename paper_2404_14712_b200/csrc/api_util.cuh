// api_util.cuh -- helpers shared by the C-ABI entry points.
#pragma once
#include "common.cuh"

namespace orbit {

int check_device();
bool valid_dtype(int dt);
bool aligned16(const void* p);

// hands out 256-byte aligned sub-buffers of a caller-provided region; with base == nullptr it only measures
struct Carver {
  char* base;
  size_t off = 0;
  explicit Carver(void* b) : base((char*)b) {}
  void* take(size_t bytes) {
    void* p = base ? (void*)(base + off) : nullptr;
    off += align_up(bytes, 256);
    return p;
  }
  template <typename T> T* take_n(size_t n) { return (T*)take(n * sizeof(T)); }
};

inline const void* offs(const void* p, size_t elems, int dt) { return (const char*)p + elems * dsize(dt); }
inline void* offs(void* p, size_t elems, int dt) { return (char*)p + elems * dsize(dt); }

}  // namespace orbit
