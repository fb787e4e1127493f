/*
 * smlm.h -- C ABI of libsmlm_b200: the data-parallel hot path of arXiv 2410.02314
 * ("An efficient inference frame for single molecule localization microscopy") for one
 * NVIDIA B200 (sm_100a).
 *
 * What the calls compute (PAPER.md = the paper text; "P:nn" = its line nn):
 *   "the image is copied into GPU memory, where the model performs inference ...
 *    post-processing is consolidated within GPU memory ... images are loaded into memory
 *    in advance, allowing the network to directly access them from specified memory
 *    locations during inference" (section 2.2, Fig. 1b);
 *   the network is a stack of dilated convolutions whose per-pixel
 *   outputs are "the probability of a fluorescent molecule, along with the offset ... of
 *   the fluorescent molecule's position relative to that pixel"; post-processing
 *   turns "these offsets into absolute coordinates" (P:192 item 3).
 * The paper gives no layer table or detection rule; sizes, activations and the rule are
 * BASELINE.json `north_star` / `configs` under the readings listed in DESIGN.md:
 *
 *   xhat = ((adu - offset) / gain) / norm_scale                              (per pixel)
 *   a0   = act(conv3x3(xhat; W0) + b0), zero padding 1, act = ReLU iff stem_relu
 *   a_{l+1} = a_l + ReLU(conv3x3 dilation d_l, zero padding d_l (a_l; W_l) + b_l)
 *   o    = Wh a_L + bh                                                       (1x1 heads)
 *   pixel q is an emitter iff sigmoid(o_p[q]) > threshold and o_p[q] beats each in-frame
 *   8-neighbour (greater, or equal with the lower linear index iy*W+ix);
 *   x_nm = (ix + xy_scale tanh(o_dx)) pixel_size, y likewise, z = z_scale tanh(o_z),
 *   photons = photon_scale softplus(o_N), bg = bg_scale softplus(o_bg), p = sigmoid(o_p).
 *
 * Every step runs in hand-written CUDA kernels; there is no CPU fallback: on a machine
 * without an sm_100 device smlm_create fails with SMLM_ERR_UNSUPPORTED_DEVICE.
 *
 * Conventions
 *   - All structs are plain data, caller-owned, copied by the callee where noted.
 *   - Status codes, never exceptions or abort().  smlm_last_error gives a message.
 *   - One smlm_ctx per host thread; calls on one ctx must not overlap.
 *   - "host" / "device" is stated for every pointer.
 */
#ifndef SMLM_H_
#define SMLM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SMLM_ABI_VERSION 4
#define SMLM_MAX_LAYERS 32

typedef struct smlm_ctx smlm_ctx; /* opaque; owns device weights, activations, staging slots, events */

typedef enum {
  SMLM_OK = 0,
  SMLM_ERR_INVALID_ARG = -1,
  SMLM_ERR_UNSUPPORTED_DEVICE = -2, /* current device is not sm_100 */
  SMLM_ERR_CUDA = -3,
  SMLM_ERR_OOM = -4,
  SMLM_ERR_OVERFLOW = -5 /* more emitters found than capacity (reported by smlm_check) */
} smlm_status;

/* Storage type of the activation maps and input type of the trunk's tensor-core MMAs.  FP16 is
 * the accuracy / throughput variant of SURVEY.md 8(f)-4: 11-bit mantissa at the same tensor
 * rate as bf16 (fp32 accumulate in both). */
enum { SMLM_FP32 = 0, SMLM_BF16 = 1, SMLM_FP16 = 2 };

/* How the windows of a tiled call (tile > 0) are formed.
 *   NONE  one window per tile x tile core (+ halo): BASELINE.json configs[3] as written.
 *   ROW   the cores of one tile row share one window (core = tile rows x the whole frame
 *         width): their x halos are computed once instead of twice.  Same emitter list. */
enum { SMLM_TILE_MERGE_NONE = 0, SMLM_TILE_MERGE_ROW = 1 };

/* K1 (uint16 unpack + normalise + 3x3 stem) kernel choice.
 *   AUTO          CUDA_CORES.  Both kernels take the same time on cfg 1 (2.2 TB/s of a_0 written inside
 *                 the step).  That is 0.41 of the write-only bandwidth of this GPU (5.4 TB/s, 16-byte
 *                 stores, measured by bench.py in the same run: profiles/bench_r3.md), so neither is at
 *                 its roof: the way the a_0 chunks are stored, not the arithmetic, sets the pace.
 *   TENSOR        the stem on the tcgen05 tensor cores (conv_chain.cu, STEM variant; 16-bit precision,
 *                 in_frames = 1): fp32 accuracy from three 16-bit pieces of every xhat and every weight,
 *                 fp32 accumulation, bias through three constant-one input channels, ReLU in the
 *                 conversion.  Half the issue slots of CUDA_CORES.  Differs from it only in summation
 *                 order (~1 fp32 ulp before the rounding of a_0 to the storage type).
 *   CUDA_CORES    stem.cu: one fp32 fmaf chain per channel, taps in (ky, kx) order (the only choice
 *                 in fp32 precision and with in_frames = 3). */
enum { SMLM_STEM_AUTO = 0, SMLM_STEM_TENSOR = 1, SMLM_STEM_CUDA_CORES = 2 };

/* Trunk convolution kernel choice for SMLM_BF16 / SMLM_FP16 (fp32 mode always uses the CUDA-core kernel). */
enum {
  SMLM_CONV_AUTO = 0,   /* tcgen05 implicit GEMM */
  SMLM_CONV_TCGEN05 = 1,
  SMLM_CONV_DIRECT = 2  /* CUDA-core kernel with the same rounding points (cross-check) */
};

/* Kernel fusion on the tcgen05 path ("post-processing is consolidated
 * within GPU memory to minimize data transfer").
 *   AUTO  HEAD + PAIRS:
 *         HEAD   the last trunk launch's epilogue evaluates the detection head of every pixel (a
 *                4 B/px logit map) and, for above-threshold pixels only, either the other heads
 *                (32-byte records) or the activations from which K3 evaluates them for the
 *                survivors of the 3x3 test; the full final map is never stored;
 *         PAIRS  consecutive trunk layers with dilations (d, 2d) run as one kernel on a
 *                thread-block cluster; the map between them stays in shared memory (C <= 48,
 *                rows of at most 1024 pixels; other layers run one per kernel).  Rows with an
 *                even number of 128-pixel segments use tcgen05 cta_group::2 (one M = 256 MMA
 *                per CTA pair, weights split between the two CTAs).
 *         K1 stays a kernel of its own (measured faster).
 *   ALL   additionally the stem (K1) is computed inside the first trunk layer's kernel when
 *         that layer is not part of a pair: a_0 never reaches HBM either.
 *   HEAD  HEAD only (every trunk layer its own kernel).
 *   PAIRS_1CTA  as AUTO with cta_group::1 MMAs in the pair kernel (the comparison twin).
 *   NONE  one kernel per step (the cross-check twin).
 * All use the same arithmetic and rounding points and give bit-identical results. */
enum { SMLM_FUSE_AUTO = 0, SMLM_FUSE_NONE = 1, SMLM_FUSE_ALL = 2, SMLM_FUSE_HEAD = 3, SMLM_FUSE_PAIRS_1CTA = 4 };

typedef struct {
  uint32_t struct_size; /* sizeof(smlm_net_desc) */
  uint32_t version;     /* SMLM_ABI_VERSION */
  int32_t channels;     /* C: multiple of 16, 16..64 */
  int32_t n_layers;     /* L: 0..SMLM_MAX_LAYERS dilated layers */
  int32_t dilations[SMLM_MAX_LAYERS]; /* d_l in 1..16 */
  int32_t head_channels; /* 5: p,dx,dy,N,bg    6: p,dx,dy,z,N,bg */
  int32_t precision;     /* SMLM_FP32 | SMLM_BF16 | SMLM_FP16 (16-bit storage + tensor-core trunk, fp32 accumulate) */
  int32_t stem_relu;     /* 1: ReLU after the stem conv */
  float norm_scale;      /* 1000 */
  float xy_scale;        /* 0.5 */
  float z_scale_nm;      /* 700 */
  float photon_scale;    /* multiplies softplus(o_N) */
  float bg_scale;        /* multiplies softplus(o_bg) */
  int32_t tile;          /* 0: whole frame; else frames are processed as tile x tile cores with a
                            halo of (receptive-field radius + 1) and detections are owned by
                            the tile whose core contains the pixel (no duplicates) */
  int32_t micro_batch;   /* frames (or tiles) per kernel launch; 0 = auto */
  int32_t conv_impl;     /* SMLM_CONV_* */
  int32_t writeback_frames; /* flush the compacted emitter list to a HOST out_emitters once
                               per this many frames, overlapped with compute (0 = library
                               default, 256; the last flush is at the end of the call) */
  int32_t fusion;        /* SMLM_FUSE_*: which steps share a kernel on the tcgen05 path */
  int32_t in_frames;     /* 0 or 1: the stem sees frame f.  3: temporal context ("contextual
                            three-frame information"): the stem is a 3 -> C convolution over the
                            normalised frames f-1, f, f+1 of the call, indices clamped to
                            [0, n_frames-1].  Not available through smlm_localize_ring. */
  int32_t tile_merge;    /* SMLM_TILE_MERGE_* */
  int32_t stem_impl;     /* SMLM_STEM_* */
} smlm_net_desc;

/* Camera model.  Scalars are used where a map pointer is NULL.  Maps are [H][W] float32,
 * HOST or DEVICE memory, read during the call (copied to the device if on the host). */
typedef struct {
  float pixel_size_nm;
  float offset; /* ADU */
  float gain;   /* ADU per photon */
  const float* offset_map;
  const float* gain_map;
} smlm_camera_params;

/* One detection, 32 bytes.  `frame` is the index within the call, `pix` = iy*W + ix in
 * full-frame coordinates. */
typedef struct {
  int32_t frame;
  int32_t pix;
  float x_nm, y_nm, z_nm; /* z_nm = 0 when head_channels == 5 */
  float photons, bg, p;
} smlm_emitter;

/*
 * smlm_create: validate `desc`, copy `weights` to the device, pre-pack the trunk weights
 * for the tensor cores.  `weights` is a HOST pointer to one little-endian fp32 blob:
 *     stem W[C][in_frames][3][3], b[C];  for l < L: W_l[C][C][3][3] (OIHW), b_l[C];  head W[n_h][C], b[n_h]
 * (cross-correlation).  Both inputs may be freed when the call returns.  Synchronous.
 * Errors: INVALID_ARG (NULL, bad sizes), UNSUPPORTED_DEVICE, CUDA, OOM.  *out_ctx = NULL on error.
 */
smlm_status smlm_create(const smlm_net_desc* desc, const void* weights, smlm_ctx** out_ctx);

/*
 * smlm_localize: the whole hot path for n_frames frames of H x W uint16.
 *   frames_u16   [n_frames][H][W], PINNED HOST memory (the preloaded ring: copied
 *                host-to-device in micro-batches on an internal copy stream, overlapped with
 *                compute) or DEVICE memory (no copy).  Pageable host memory is refused
 *                (INVALID_ARG).  Must stay valid until `cuda_stream` has finished the call.
 *   camera       HOST struct, copied.
 *   threshold    detection threshold on p (strict >).  <= 0: every local maximum; >= 1: none.
 *   out_emitters DEVICE or PINNED HOST array with room for `*out_count` records.  Order of
 *                records is unspecified (atomic compaction); compare as a set.
 *   out_count    HOST pointer.  In: capacity of out_emitters in records.  Out: number of
 *                emitters found (may exceed the capacity; only the first `capacity` in arrival
 *                order are stored).  Written asynchronously, from a host callback ordered on the
 *                stream: the int64 must stay allocated until the stream has finished the call (do
 *                not pass the address of a temporary), and it is valid from then on.
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream).  The call only enqueues work;
 *                it is ordered after earlier work on that stream; results are valid once the
 *                stream has been synchronised.
 * Errors: INVALID_ARG, CUDA, OOM synchronously; overflow via smlm_check after the sync.
 */
smlm_status smlm_localize(smlm_ctx* ctx, const uint16_t* frames_u16, int64_t n_frames, int32_t H,
                          int32_t W, const smlm_camera_params* camera, float threshold,
                          smlm_emitter* out_emitters, int64_t* out_count, void* cuda_stream);

/* After the stream of the last smlm_localize has been synchronised: SMLM_ERR_OVERFLOW if it
 * found more emitters than the capacity, SMLM_ERR_CUDA if an asynchronous error is pending. */
smlm_status smlm_check(smlm_ctx* ctx);

/*
 * The preload ring fed from storage ("multiple processes handle data loading and network
 * inference simultaneously"; "images are loaded in advance into specified memory
 * locations"; the NVMe -> GPU experiment of P:196-198).
 *   smlm_ring_open: `path` is a raw little-endian uint16 file holding [n_frames][H][W] at
 *     `byte_offset`.  `n_threads` reader threads (pread) fill a ring of `n_slots` >= 2 chunks of
 *     `chunk_frames` frames in PINNED host memory, in file order, as slots become free.
 *     flags: SMLM_RING_PAGEABLE allocates the ring with malloc (host-logic tests on a machine
 *     without a GPU; smlm_localize_ring refuses such a ring).
 *     Errors: INVALID_ARG (bad sizes, file missing or too short), CUDA (pinned allocation), OOM.
 *   smlm_localize_ring: smlm_localize over the whole file.  Chunk k is localized from ring slot
 *     k % n_slots (H2D on the ctx's copy stream) while the readers fill the following slots;
 *     a slot is handed back to the readers when its last H2D copy has finished.  `frame` of
 *     the records is the index in the file; one emitter list, same arguments and error
 *     behaviour as smlm_localize.  Enqueues GPU work asynchronously but BLOCKS the calling
 *     host thread while it waits for the disk.  The ring is rewound first, so it can be used
 *     for several passes.
 *   smlm_ring_acquire / smlm_ring_release: the consumer side by hand (tests, custom loops):
 *     acquire blocks until the next chunk is in memory (*n_frames = 0 at the end of the file),
 *     release(first_frame) lets the readers refill its slot.
 *   smlm_ring_rewind: start over at the first chunk (what smlm_localize_ring does on entry), also
 *     after a pass that was abandoned part-way.  Blocks until every chunk handed out so far has
 *     been released - release what you acquired first - and until reads in flight have ended.
 *     Not to be called concurrently with acquire / release / smlm_localize_ring on the same ring.
 *   smlm_ring_close: stops the readers, frees the ring.  NULL is allowed.  GPU work of an earlier
 *     smlm_localize_ring on this ring must have finished (synchronise its stream first): that
 *     work hands slots back to the ring from stream callbacks.
 */
typedef struct smlm_ring smlm_ring;
enum { SMLM_RING_PAGEABLE = 1 };
smlm_status smlm_ring_open(const char* path, int64_t byte_offset, int64_t n_frames, int32_t H, int32_t W,
                           int32_t chunk_frames, int32_t n_slots, int32_t n_threads, int32_t flags,
                           smlm_ring** out_ring);
smlm_status smlm_localize_ring(smlm_ctx* ctx, smlm_ring* ring, const smlm_camera_params* camera,
                               float threshold, smlm_emitter* out_emitters, int64_t* out_count,
                               void* cuda_stream);
smlm_status smlm_ring_acquire(smlm_ring* ring, const uint16_t** frames, int64_t* n_frames,
                              int64_t* first_frame);
smlm_status smlm_ring_release(smlm_ring* ring, int64_t first_frame);
smlm_status smlm_ring_rewind(smlm_ring* ring);
void smlm_ring_close(smlm_ring* ring);

/* Synchronise, free everything the ctx owns.  NULL is allowed. */
void smlm_destroy(smlm_ctx* ctx);

/* Message of the last error on this ctx (or of the last failed smlm_create when ctx is NULL).
 * The pointer stays valid until the next call on the ctx. */
const char* smlm_last_error(const smlm_ctx* ctx);

/* Number of kernel launches this ctx has enqueued so far (bench.py's `gpu_launches`). */
int64_t smlm_launch_count(const smlm_ctx* ctx);

/* Per-kernel timing for bench.py's roofline: when enabled, every launch of K1 (stem), K2
 * (trunk convolution) and K3 (heads + post-processing) is bracketed by CUDA events on the
 * launching stream; smlm_kernel_time_ms (after a stream sync) sums the launches of one kind
 * since timing was last enabled.  Disabled by default: the events cost ~1 us each and switch
 * off the programmatic overlap between consecutive layers. */
/* CONV: one trunk layer per launch; CONV_PAIR: two trunk layers per launch (SMLM_FUSE_* PAIRS). */
enum { SMLM_KERNEL_STEM = 0, SMLM_KERNEL_CONV = 1, SMLM_KERNEL_POST = 2, SMLM_KERNEL_CONV_PAIR = 3 };
smlm_status smlm_kernel_timing(smlm_ctx* ctx, int32_t enable);
smlm_status smlm_kernel_time_ms(smlm_ctx* ctx, int32_t kind, double* total_ms, int64_t* launches);

/*
 * Test/debug exports.  BASELINE.json asks for parity on the raw output maps, which the
 * production path never writes to memory; these two calls expose them.
 *   smlm_debug_forward_maps: `maps` is DEVICE float32 [n][n_h][H][W], the PRE-activation
 *     head outputs o.  `trunk` (may be NULL) is DEVICE float32 [n][L+1][H][W][C], a_0..a_L.
 *     frames_u16 as in smlm_localize.  Whole frames only (tile is ignored).
 *   smlm_debug_postprocess: runs detection + decode + compaction on caller-supplied
 *     DEVICE float32 maps o [n][n_h][H][W].
 */
smlm_status smlm_debug_forward_maps(smlm_ctx* ctx, const uint16_t* frames_u16, int64_t n_frames,
                                    int32_t H, int32_t W, const smlm_camera_params* camera,
                                    float* maps, float* trunk, void* cuda_stream);
smlm_status smlm_debug_postprocess(smlm_ctx* ctx, const float* maps, int64_t n_frames, int32_t H,
                                   int32_t W, const smlm_camera_params* camera, float threshold,
                                   smlm_emitter* out_emitters, int64_t* out_count, void* cuda_stream);

/* Measurement aid for bench.py (no part of the method): fill `bytes` (a multiple of 16) of DEVICE
 * memory at `dst` (16-byte aligned) with a byte pattern.  mode 0: cudaMemsetAsync; mode 1: a kernel
 * of 16-byte stores.  Asynchronous on `cuda_stream`.  The write-only bandwidth K1 is held against. */
smlm_status smlm_debug_fill(void* dst, int64_t bytes, int32_t mode, void* cuda_stream);

/*
 * smlm_postprocess_static: post-processing for callers that cannot allocate GPU memory.
 *
 * Who this is for.  All calls above work on an smlm_ctx, and a ctx allocates: smlm_create calls
 * cudaMalloc, and smlm_localize / smlm_debug_postprocess call it again when a frame size or a
 * capacity grows.  Some programs cannot have that happen under them:
 *   - a live acquisition loop, where cudaMalloc / cudaFree would stall the whole device (both wait
 *     for running work) while the camera's next frames are being copied in;
 *   - a plug-in or custom operator inside a host application that reserved the GPU's memory for
 *     its own pool and only hands out buffers - a cudaMalloc from inside it can simply fail;
 *   - a process that must do all its allocation at start-up.
 * This one call needs no ctx and calls no cudaMalloc, cudaFree, cudaMallocHost or any library
 * routine that allocates.  The caller passes the maps and the output list; the bookkeeping of the
 * compaction lives in a fixed array of SMLM_POST_STATIC_SCRATCH_BYTES (1 MiB) that is part of the
 * library's device code: every GPU on which the library is used holds that 1 MiB from the moment
 * its code is loaded there until the process exits.
 *
 * What it computes: the same rule as smlm_debug_postprocess (threshold on sigmoid(o_p), 3x3 local
 * maximum with the lower-index tie rule, decode of the other heads; formulas at the top of this
 * file) on caller-supplied pre-activation maps.  Same records, but in a FIXED order: by frame,
 * then by 32 x 64 pixel tile (tile rows top to bottom, tiles left to right), then row-major
 * inside the tile.  Two calls on the same input give byte-identical lists.
 *
 *   maps         DEVICE float32 [n_frames][head_channels][H][W], pre-activation head outputs o.
 *   params       HOST struct, read during the call.
 *   threshold    as in smlm_localize.
 *   out_emitters DEVICE (or pinned host) array of `capacity` records, 16-byte aligned; may be NULL
 *                when capacity == 0 (count only).  Of more than `capacity` detections the first
 *                `capacity` in the order above are stored.
 *   out_count    DEVICE (or pinned host) int64 the GPU can write: number of detections found (may
 *                exceed capacity).  Valid once the stream has finished.  Unlike smlm_localize this
 *                is not a pageable host pointer: forwarding to one would need a host allocation.
 *   cuda_stream  a cudaStream_t (NULL = legacy default stream); the call only enqueues three kernels.
 *
 * Size limit: ceil(H/32) * ceil(W/64) * n_frames <= SMLM_POST_STATIC_MAX_TILES (262 080 tiles:
 * 8 190 frames of 256 x 256, 2 047 of 512 x 512, 127 of 2048 x 2048).  A larger call is refused
 * with SMLM_ERR_INVALID_ARG and a message that names the limit; split it by frames.
 *
 * First call on a device: looks up the device address of the scratch array (cudaGetSymbolAddress,
 * with that device current - the current device of the calling thread is the one used) and keeps
 * it for later calls.  That lookup may make the CUDA runtime load the library's device code on
 * that GPU, so make the first call on each device during start-up, before any stream capture
 * begins.  The lookup and all argument checks are thread-safe.
 *
 * Sharing: all calls on one device use the same array.  Nothing needs clearing between calls
 * (each call overwrites every word before it reads it), but calls whose kernels can run at the
 * same time on one GPU - different streams, or several host threads - race on it and produce
 * wrong lists.  Keep calls on one device in one stream, or order them with events.
 *
 * Errors (synchronous): INVALID_ARG (NULL, sizes, the limit above, head_channels not 5 / 6),
 * UNSUPPORTED_DEVICE (current device is not sm_100), CUDA.  smlm_postprocess_static_error returns
 * the message of the last failed call on the calling thread (valid until that thread's next call).
 */
#define SMLM_POST_STATIC_SCRATCH_BYTES 1048576
#define SMLM_POST_STATIC_MAX_TILES 262080 /* (SCRATCH_BYTES - 256) / 4 */
typedef struct {
  int32_t head_channels; /* 5: p,dx,dy,N,bg    6: p,dx,dy,z,N,bg */
  float xy_scale, z_scale_nm, photon_scale, bg_scale; /* as in smlm_net_desc */
  float pixel_size_nm;                                /* as in smlm_camera_params */
} smlm_post_params;
smlm_status smlm_postprocess_static(const float* maps, int64_t n_frames, int32_t H, int32_t W,
                                    const smlm_post_params* params, float threshold,
                                    smlm_emitter* out_emitters, int64_t capacity, int64_t* out_count,
                                    void* cuda_stream);
const char* smlm_postprocess_static_error(void);

#ifdef __cplusplus
}
#endif
#endif /* SMLM_H_ */
