// The preload ring of the paper's inference frame ("multiple processes handle data
// loading and network inference simultaneously", "images are loaded in advance into
// specified memory locations"; the disk -> GPU experiment of P:196-198): reader threads fill
// a ring of pinned host chunks from a raw frame file while the GPU works on earlier chunks.
// Host code only; nothing here is shared with oracle/.
#pragma once
#include <stdint.h>

#include <atomic>
#include <condition_variable>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

struct smlm_ring {
  int fd = -1;
  int64_t byte_offset = 0, n_frames = 0;
  int H = 0, W = 0, chunk_frames = 0, n_slots = 0;
  bool pinned = false;
  int64_t n_chunks = 0;
  uint16_t* buf = nullptr;  // n_slots x chunk_frames x H x W

  // chunk k lives in slot k % n_slots.  loaded[s] = index of the chunk the slot holds (-1:
  // none); free_from[s] = first chunk index that may be loaded into the slot (advanced by
  // n_slots on release), so chunks enter a slot strictly in order.
  std::mutex mu;
  std::condition_variable cv;
  std::vector<int64_t> loaded, free_from;
  std::atomic<int64_t> next_chunk{0};
  int64_t next_acquire = 0;
  int64_t gen = 0;       // bumped by a rewind: readers drop the chunk they were assigned before it
  int active_reads = 0;  // readers inside pread
  bool rewinding = false;  // a rewind is between its generation bump and its reset: readers stay parked
  bool touched = false;  // a chunk has been handed out since the last rewind
  int64_t outstanding = 0;  // chunks handed out and not yet released (a rewind waits for them)
  int64_t by_hand = 0;      // ... of which through smlm_ring_acquire
  bool stop = false;
  std::string error;
  std::vector<std::thread> readers;

  size_t slot_elems() const { return (size_t)chunk_frames * H * W; }
  int64_t frames_of(int64_t k) const {
    int64_t lo = k * chunk_frames;
    return n_frames - lo < chunk_frames ? n_frames - lo : chunk_frames;
  }
};

namespace smlm {
// blocks until chunk `k` is in memory; returns its address or nullptr (ring->error is set)
const uint16_t* ring_wait_chunk(smlm_ring* r, int64_t k);
// the slot of chunk k may be refilled (with chunk k + n_slots)
void ring_release_chunk(smlm_ring* r, int64_t k);
// all chunks start over (a ring can serve several passes over the file).  Blocks until every
// chunk handed out so far has been released: the previous pass's asynchronous H2D copies still
// read the slots, and a release that arrived after the rewind would free a slot of the new pass.
void ring_rewind(smlm_ring* r);
}  // namespace smlm
