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

// shape / dtype / flag checks shared by orbit_block_* (api_block.cu) and the rank-local orbit_rank_* calls (api_shard.cu)
int check_block(const orbit_block_desc* d);
int check_block_params(const orbit_block_desc* d, const orbit_block_params* P);   // reads P->shards[0 .. T)
int check_shard_params(const orbit_block_desc* d, const orbit_block_params* P);   // reads P->shards[0] only

inline const void* offs(const void* p, size_t elems, int dt) { return (const char*)p + elems * dsize(dt); }
inline void* offs(void* p, size_t elems, int dt) { return (char*)p + elems * dsize(dt); }

}  // namespace orbit
