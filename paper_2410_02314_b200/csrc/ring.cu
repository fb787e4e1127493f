// Reader threads + pinned ring (ring.cuh) and its C ABI (include/smlm.h: smlm_ring_*).
#include "ring.cuh"

#include <cuda_runtime.h>
#include <errno.h>
#include <fcntl.h>
#include <string.h>
#include <sys/stat.h>
#include <unistd.h>

#include <new>

#include "../../include/smlm.h"

namespace smlm {

namespace {

void reader_main(smlm_ring* r) {
  for (;;) {
    int64_t k, g;
    {
      std::unique_lock<std::mutex> lk(r->mu);
      // parked while the file is exhausted, and for the WHOLE of a rewind: an assignment taken
      // between the rewind's generation bump and its reset of next_chunk / free_from would carry
      // the new generation with an old chunk index and be read twice
      r->cv.wait(lk, [&] { return r->stop || (!r->rewinding && r->next_chunk.load() < r->n_chunks); });
      if (r->stop) return;
      k = r->next_chunk.load();
      g = r->gen;
      r->next_chunk.store(k + 1);
      const int s = (int)(k % r->n_slots);
      r->cv.wait(lk, [&] { return r->stop || r->gen != g || r->free_from[s] == k; });
      if (r->stop) return;
      if (r->gen != g) continue;  // rewound while waiting: this assignment is void
      ++r->active_reads;
    }
    const int s = (int)(k % r->n_slots);
    uint8_t* dst = reinterpret_cast<uint8_t*>(r->buf + (size_t)s * r->slot_elems());
    size_t want = (size_t)r->frames_of(k) * r->H * r->W * sizeof(uint16_t);
    off_t off = (off_t)(r->byte_offset + k * (int64_t)r->slot_elems() * (int64_t)sizeof(uint16_t));
    std::string err;
    while (want > 0) {
      ssize_t got = pread(r->fd, dst, want, off);
      if (got < 0 && errno == EINTR) continue;
      if (got <= 0) {
        err = got == 0 ? "unexpected end of the frame file" : std::string("pread: ") + strerror(errno);
        break;
      }
      dst += got;
      off += got;
      want -= (size_t)got;
    }
    {
      std::lock_guard<std::mutex> lk(r->mu);
      --r->active_reads;
      if (!err.empty()) {
        r->error = err;
        r->stop = true;
      } else if (r->gen == g) {
        r->loaded[s] = k;
      }
    }
    r->cv.notify_all();
  }
}

}  // namespace

const uint16_t* ring_wait_chunk(smlm_ring* r, int64_t k) {
  const int s = (int)(k % r->n_slots);
  std::unique_lock<std::mutex> lk(r->mu);
  r->touched = true;
  r->cv.wait(lk, [&] { return r->stop || r->loaded[s] == k; });
  if (r->loaded[s] != k) return nullptr;
  ++r->outstanding;
  return r->buf + (size_t)s * r->slot_elems();
}

void ring_release_chunk(smlm_ring* r, int64_t k) {
  const int s = (int)(k % r->n_slots);
  {
    std::lock_guard<std::mutex> lk(r->mu);
    if (r->loaded[s] == k) {
      r->loaded[s] = -1;
      r->free_from[s] = k + r->n_slots;
      --r->outstanding;
    }
  }
  r->cv.notify_all();
}

// Start over at chunk 0.  Nothing to do on a ring no chunk of which has been handed out; else
// wait until every chunk handed out has been released (smlm_localize_ring releases from a
// callback of its copy stream: the host may be several calls ahead of the GPU, the previous
// pass's copies still read the slots, and a late release of old chunk k would otherwise free
// the slot that holds new chunk k - the host then waits for that chunk forever), void the
// readers' pending assignments (generation bump) and wait for reads in flight, so that no
// stale reader writes into a slot of the new pass.  The mutex is released inside those waits:
// `rewinding` keeps the readers parked until next_chunk / free_from / loaded are reset.
void ring_rewind(smlm_ring* r) {
  {
    std::unique_lock<std::mutex> lk(r->mu);
    if (!r->touched) return;
    r->cv.wait(lk, [&] { return r->stop || r->outstanding == 0; });
    r->rewinding = true;  // readers take no assignment until the reset below is complete
    ++r->gen;
    r->cv.notify_all();
    r->cv.wait(lk, [&] { return r->stop || r->active_reads == 0; });
    for (int s = 0; s < r->n_slots; ++s) {
      r->loaded[s] = -1;
      r->free_from[s] = s;
    }
    r->next_chunk.store(0);
    r->next_acquire = 0;
    r->touched = false;
    r->rewinding = false;
  }
  r->cv.notify_all();
}

}  // namespace smlm

extern "C" {

smlm_status smlm_ring_open(const char* path, int64_t byte_offset, int64_t n_frames, int32_t H, int32_t W,
                           int32_t chunk_frames, int32_t n_slots, int32_t n_threads, int32_t flags,
                           smlm_ring** out) {
  if (out) *out = nullptr;
  if (!path || !out || byte_offset < 0 || n_frames < 0 || H < 1 || W < 1 || chunk_frames < 1 || n_slots < 2 ||
      n_threads < 1 || n_threads > 64 || (flags & ~SMLM_RING_PAGEABLE))
    return SMLM_ERR_INVALID_ARG;
  smlm_ring* r = new (std::nothrow) smlm_ring;
  if (!r) return SMLM_ERR_OOM;
  r->fd = open(path, O_RDONLY);
  if (r->fd < 0) {
    delete r;
    return SMLM_ERR_INVALID_ARG;
  }
  struct stat sb;
  if (fstat(r->fd, &sb) != 0 ||
      (int64_t)sb.st_size < byte_offset + n_frames * (int64_t)H * W * (int64_t)sizeof(uint16_t)) {
    close(r->fd);
    delete r;
    return SMLM_ERR_INVALID_ARG;  // the file is shorter than n_frames frames
  }
  r->byte_offset = byte_offset;
  r->n_frames = n_frames;
  r->H = H;
  r->W = W;
  r->chunk_frames = chunk_frames;
  r->n_slots = n_slots;
  r->n_chunks = (n_frames + chunk_frames - 1) / chunk_frames;
  r->pinned = !(flags & SMLM_RING_PAGEABLE);
  const size_t bytes = (size_t)n_slots * r->slot_elems() * sizeof(uint16_t);
  if (r->pinned) {
    if (cudaHostAlloc(reinterpret_cast<void**>(&r->buf), bytes, cudaHostAllocDefault) != cudaSuccess) {
      cudaGetLastError();
      close(r->fd);
      delete r;
      return SMLM_ERR_CUDA;
    }
  } else {
    r->buf = static_cast<uint16_t*>(malloc(bytes));
    if (!r->buf) {
      close(r->fd);
      delete r;
      return SMLM_ERR_OOM;
    }
  }
  r->loaded.assign(n_slots, -1);
  r->free_from.resize(n_slots);
  for (int s = 0; s < n_slots; ++s) r->free_from[s] = s;
  for (int t = 0; t < n_threads; ++t) r->readers.emplace_back(smlm::reader_main, r);
  *out = r;
  return SMLM_OK;
}

void smlm_ring_close(smlm_ring* r) {
  if (!r) return;
  {
    std::lock_guard<std::mutex> lk(r->mu);
    r->stop = true;
  }
  r->cv.notify_all();
  for (auto& t : r->readers) t.join();
  if (r->buf) {
    if (r->pinned) cudaFreeHost(r->buf);
    else free(r->buf);
  }
  if (r->fd >= 0) close(r->fd);
  delete r;
}

smlm_status smlm_ring_acquire(smlm_ring* r, const uint16_t** frames, int64_t* n_frames, int64_t* first_frame) {
  if (!r || !frames || !n_frames) return SMLM_ERR_INVALID_ARG;
  *frames = nullptr;
  *n_frames = 0;
  const int64_t k = r->next_acquire;
  if (k >= r->n_chunks) return SMLM_OK;  // end of the file: *n_frames = 0
  const uint16_t* p = smlm::ring_wait_chunk(r, k);
  if (!p) return SMLM_ERR_INVALID_ARG;
  *frames = p;
  *n_frames = r->frames_of(k);
  if (first_frame) *first_frame = k * r->chunk_frames;
  r->next_acquire = k + 1;
  {
    std::lock_guard<std::mutex> lk(r->mu);
    ++r->by_hand;
  }
  return SMLM_OK;
}

smlm_status smlm_ring_rewind(smlm_ring* r) {
  if (!r) return SMLM_ERR_INVALID_ARG;
  smlm::ring_rewind(r);
  std::lock_guard<std::mutex> lk(r->mu);
  return r->stop ? SMLM_ERR_INVALID_ARG : SMLM_OK;  // a read error stopped the ring
}

smlm_status smlm_ring_release(smlm_ring* r, int64_t first_frame) {
  if (!r || first_frame < 0 || first_frame % r->chunk_frames) return SMLM_ERR_INVALID_ARG;
  {
    std::lock_guard<std::mutex> lk(r->mu);
    const int64_t k = first_frame / r->chunk_frames;
    if (r->loaded[(size_t)(k % r->n_slots)] == k && r->by_hand > 0) --r->by_hand;
  }
  smlm::ring_release_chunk(r, first_frame / r->chunk_frames);
  return SMLM_OK;
}

}  // extern "C"
