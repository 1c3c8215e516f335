// Stream-ordered device memory pool (§3.2 "Memory Arenas":
// allocate in large chunks and hand out pieces, first fit, so that steady-state time steps make
// no cudaMalloc / cudaFree calls). All memory handed out is used on ONE stream, so a freed block
// may be reused at once: any later use is ordered after the earlier one by the stream itself.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <map>
#include <vector>

namespace pic {

class Pool {
 public:
  explicit Pool(size_t min_chunk = (size_t)64 << 20) : min_chunk_(min_chunk) {}
  ~Pool() { release(); }
  Pool(const Pool&) = delete;
  Pool& operator=(const Pool&) = delete;

  // nullptr on failure (cudaMalloc error is cleared and kept in last_error())
  void* alloc(size_t bytes) {
    if (bytes == 0) bytes = 1;
    bytes = (bytes + kAlign - 1) / kAlign * kAlign;
    for (auto it = free_.begin(); it != free_.end(); ++it) {   // first fit, address order
      if (it->second >= bytes) {
        char* p = it->first;
        size_t rest = it->second - bytes;
        free_.erase(it);
        if (rest) free_[p + bytes] = rest;
        used_[p] = bytes;
        in_use_ += bytes;
        return p;
      }
    }
    size_t chunk = bytes > min_chunk_ ? bytes : min_chunk_;
    void* base = nullptr;
    cudaError_t e = cudaMalloc(&base, chunk);
    if (e != cudaSuccess && chunk > bytes) {   // a smaller chunk may still fit
      cudaGetLastError();
      chunk = bytes;
      e = cudaMalloc(&base, chunk);
    }
    if (e != cudaSuccess) {
      last_error_ = e;
      cudaGetLastError();
      return nullptr;
    }
    chunks_.push_back({(char*)base, chunk});
    held_ += chunk;
    n_chunks_++;
    if (chunk > bytes) free_[(char*)base + bytes] = chunk - bytes;
    used_[(char*)base] = bytes;
    in_use_ += bytes;
    return base;
  }

  // One chunk of at least `bytes`, added to the free list (no-op if that much is free in one block already):
  // a caller that knows what it is about to allocate asks for it in ONE cudaMalloc instead of one per array
  // (pic_add_species: 25 arrays, 2.6 GB on C2 — cudaMalloc is a synchronising driver call of ~ 0.3 ms each).
  // Failure is not an error here: the allocations that follow fall back to their own chunks.
  void reserve(size_t bytes) {
    bytes = (bytes + kAlign - 1) / kAlign * kAlign;
    for (auto& f : free_)
      if (f.second >= bytes) return;
    if (bytes < min_chunk_) bytes = min_chunk_;
    void* base = nullptr;
    if (cudaMalloc(&base, bytes) != cudaSuccess) {
      cudaGetLastError();
      return;
    }
    chunks_.push_back({(char*)base, bytes});
    held_ += bytes;
    n_chunks_++;
    free_[(char*)base] = bytes;
  }

  void free(void* ptr) {
    if (!ptr) return;
    auto u = used_.find((char*)ptr);
    if (u == used_.end()) return;
    char* p = u->first;
    size_t n = u->second;
    used_.erase(u);
    in_use_ -= n;
    auto next = free_.lower_bound(p);
    // merge with the following free block if adjacent and in the same chunk
    if (next != free_.end() && p + n == next->first && same_chunk(p, next->first)) {
      n += next->second;
      next = free_.erase(next);
    }
    if (next != free_.begin()) {
      auto prev = std::prev(next);
      if (prev->first + prev->second == p && same_chunk(prev->first, p)) {
        prev->second += n;
        return;
      }
    }
    free_[p] = n;
  }

  void release() {
    for (auto& c : chunks_) cudaFree(c.base);
    chunks_.clear(); free_.clear(); used_.clear();
    held_ = in_use_ = 0;
  }

  int64_t n_chunks() const { return n_chunks_; }      // cudaMalloc calls so far
  size_t bytes_held() const { return held_; }
  size_t bytes_in_use() const { return in_use_; }
  cudaError_t last_error() const { return last_error_; }

 private:
  static constexpr size_t kAlign = 512;
  struct Chunk { char* base; size_t size; };
  bool same_chunk(char* a, char* b) const {
    for (auto& c : chunks_)
      if (a >= c.base && a < c.base + c.size) return b >= c.base && b < c.base + c.size;
    return false;
  }
  size_t min_chunk_;
  std::vector<Chunk> chunks_;
  std::map<char*, size_t> free_;   // address -> size
  std::map<char*, size_t> used_;
  size_t held_ = 0, in_use_ = 0;
  int64_t n_chunks_ = 0;
  cudaError_t last_error_ = cudaSuccess;
};

}  // namespace pic
