/*
 * aceapex.h — C-ABI of the B200-native (sm_100a) two-layer block decoder.
 *
 * The operation is the one arxiv/paper_2606_24531 states as its problem: decode the output of
 * a two-layer codec — an entropy layer applied per fixed-size block (per-block
 * ANS; :124 ref [6] interleaved rANS) under a match layer whose back-references are absolute
 * positions in the decompressed output — either whole, for a
 * set of blocks (PAPER.md:104 range decode), or for the one block named by a single coordinate
 * ("unified seek"), bit-perfect and without touching any other block
 * (PAPER.md:49-51). The container layout is this build's own (FORMAT.md): the paper fixes none
 * (PAPER.md:110).
 *
 * Conventions
 *   - Every pointer is tagged in its comment as DEVICE (CUDA global memory of the current
 *     device) or HOST. The library never allocates, frees or keeps ownership of caller buffers;
 *     `d_container` and the scratch buffer must outlive the context.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Return value: ACEAPEX_OK (0) or a negative ACEAPEX_E_* code. No exceptions, no aborts.
 *   - Argument errors are reported synchronously by the call. Violations found on the device
 *     while decoding (a corrupt record, a reference that is not strictly before its own
 *     position, ...) never cause an out-of-bounds access: the offending block is left
 *     unwritten, a sticky status word is set in device memory and aceapex_device_status()
 *     returns ACEAPEX_E_CORRUPT.
 *   - Every decode call is asynchronous on `cuda_stream`: decode_all / decode_range enqueue two
 *     kernels per batch of n_slots blocks (decode_range with first > 0: three), decode_blocks / seek
 *     one fused kernel per group of n_targets blocks (the copy-hop loop runs on the device and ends
 *     there; no host read-back).
 *   - There is no CPU fallback: without a CUDA device every call except aceapex_strerror and
 *     aceapex_version fails with ACEAPEX_E_CUDA.
 */
#ifndef ACEAPEX_H
#define ACEAPEX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
    ACEAPEX_OK = 0,
    ACEAPEX_E_ARG = -1,       /* NULL / misaligned / inconsistent argument */
    ACEAPEX_E_FORMAT = -2,    /* bad magic, version or header field (FORMAT.md section 1) */
    ACEAPEX_E_CAPACITY = -3,  /* output or scratch buffer too small */
    ACEAPEX_E_CORRUPT = -4,   /* container violates a validity rule (FORMAT.md sections 2-4) */
    ACEAPEX_E_RANGE = -5,     /* block id or coordinate outside the decompressed output */
    ACEAPEX_E_NOMEM = -6,     /* host allocation failed */
    ACEAPEX_E_CUDA = -7,      /* a CUDA runtime call failed (no device, launch error, ...) */
    ACEAPEX_E_STATE = -8      /* call order: scratch not set */
};

/* aceapex_decode_blocks flags: where block ids[i] lands in d_out */
enum {
    ACEAPEX_PACKED = 0,       /* at d_out + i * 16384 */
    ACEAPEX_ABSOLUTE = 1      /* at d_out + ids[i] * 16384 (its position in the full output) */
};

typedef struct aceapex_ctx aceapex_ctx; /* opaque */

typedef struct {
    uint64_t total_len;      /* decompressed bytes */
    uint64_t n_blocks;       /* ceil(total_len / 16384) */
    uint64_t container_bytes;
    uint32_t block_size;     /* 16384 (a library built with -DACEAPEX_BLOCK_LOG2=12..15 for the block-size sweep: 4096 .. 32768;
                                every "16384" below then reads as this value) */
    uint32_t offset_width;   /* 4 or 8 */
    uint32_t max_depth;      /* header promise D (0 = none) */
    uint32_t window;         /* header promise R (0 = none) */
    uint32_t max_level;      /* largest in-block tag */
    uint32_t max_n_seq;      /* largest n_seq of any block record (found by the open-time scan) */
} aceapex_info;

/* Library version (major*10000 + minor*100 + patch). */
int aceapex_version(void);

/* Open a container that already resides in device memory.
 *   d_container  DEVICE, 16-byte aligned, `nbytes` bytes, FORMAT.md section 1; caller-owned and
 *                must stay valid and unmodified until aceapex_close.
 *   h_header     HOST, optional: the first 64 bytes of the container (or more; only 64 are
 *                read). NULL = the library copies the header from the device.
 *   out          HOST, receives the context.
 * Validates the header (ACEAPEX_E_FORMAT) and runs one device pass over all block-record
 * headers (one entropy entry point per block) that checks them and finds the
 * largest n_seq; synchronises the device. A corrupt record header yields ACEAPEX_E_CORRUPT.  * ACEAPEX_E_CAPACITY: the container's densest block needs more shared memory in the match kernel than the device
 * offers (only reachable with 32 KiB blocks holding more than about 6,000 sequences). */
int aceapex_open(const void *d_container, size_t nbytes, const void *h_header, aceapex_ctx **out);

/* HOST out. */
int aceapex_info_get(const aceapex_ctx *ctx, aceapex_info *out);

/* Scratch the caller must provide (DEVICE, 256-byte aligned) for the given batch limits.
 *   n_slots    decoded-token slots: blocks whose token streams are resident at once. decode_all
 *              works through the container in batches of n_slots blocks; decode_blocks / seek
 *              use one slot per distinct block touched by a group of targets (with fewer slots
 *              they still decode correctly, in several rounds). >= 1.
 *   n_targets  target blocks whose per-byte chase state is resident at once in decode_blocks
 *              (the id list is processed in groups of n_targets); 0 if only decode_all is used.
 * Returns 0 on a NULL context. */
size_t aceapex_scratch_bytes(const aceapex_ctx *ctx, size_t n_slots, size_t n_targets);

/* Hand the scratch buffer to the context (caller keeps ownership; must outlive the context or
 * the next set_scratch). `nbytes` must be >= aceapex_scratch_bytes(ctx, n_slots, n_targets).
 * Enqueues one memset on `cuda_stream`. */
int aceapex_set_scratch(aceapex_ctx *ctx, void *d_scratch, size_t nbytes, size_t n_slots,
                        size_t n_targets, void *cuda_stream);

/* Full two-layer decode: writes d_out[0, total_len) and nothing else.
 *   d_out  DEVICE, capacity `out_capacity` >= total_len (else ACEAPEX_E_CAPACITY). 16-byte
 *          alignment enables the vector store path; any alignment is accepted.
 * Every block is entropy-decoded (32-lane rANS per stream, FORMAT.md section 3) and rebuilt from
 * its literals plus copies from absolute output positions (FORMAT.md section 4); a block that
 * copies from earlier blocks waits until those are complete ("any block decodes
 * once the blocks holding its source bytes are present"). */
int aceapex_decode_all(aceapex_ctx *ctx, void *d_out, size_t out_capacity, void *cuda_stream);

/* Range decode ("makes range decoding mandatory rather than optional": blocks 0-1000 of a 3 M block
 * archive; a file decoded in sub-batches): blocks [first, first + count) through both layers into a
 * RANGE-SIZED buffer, block first + i at d_out + i * 16384; writes d_out[0, (count-1)*16384 + block_len(last)) and
 * nothing else.
 *   first, count  blocks; first + count <= n_blocks (else ACEAPEX_E_RANGE); count == 0 is a no-op.
 *   d_out         DEVICE, capacity `out_capacity` >= the bytes written (else ACEAPEX_E_CAPACITY).
 * The range runs through the same entropy and match kernels as aceapex_decode_all, in sub-batches of
 * min(n_slots, n_targets) blocks. Copies whose source starts below block `first` cannot be taken from the buffer:
 * exactly those bytes are first followed to their origins through the compressed data (the isolated path of
 * aceapex_decode_blocks, restricted to them) and written in place; needs n_targets >= 1 in the scratch when
 * first > 0 (else ACEAPEX_E_STATE). Asynchronous on `cuda_stream`. */
int aceapex_decode_range(aceapex_ctx *ctx, uint64_t first, uint64_t count, void *d_out, size_t out_capacity,
                         void *cuda_stream);

/* Isolated decode of the listed blocks.
 *   h_ids  HOST, n_ids block ids, each < n_blocks (else ACEAPEX_E_RANGE); duplicates allowed.
 *   d_out  DEVICE. PACKED: block ids[i] -> d_out[i*16384, i*16384 + block_len(ids[i])),
 *          capacity >= n_ids*16384 - (16384 - block_len(last listed id)) is NOT assumed: the
 *          required capacity is the end of the last byte written. ABSOLUTE: block ids[i] ->
 *          d_out[ids[i]*16384, ...), capacity >= end of the highest listed block.
 * Isolation contract: only the byte ranges of the listed blocks are written in
 * d_out; every source byte that lives in another block is re-derived from the compressed data
 * (origin chase through absolute offsets, SURVEY.md section 8c reading A7) inside the scratch. */
int aceapex_decode_blocks(aceapex_ctx *ctx, const uint64_t *h_ids, size_t n_ids, void *d_out,
                          size_t out_capacity, uint32_t flags, void *cuda_stream);

/* Unified seek: `coord` is an absolute byte offset in the decompressed
 * output (coord >= total_len -> ACEAPEX_E_RANGE); the enclosing block b = coord >> 14 is decoded
 * in isolation into d_dst[0, block_len).
 *   d_dst            DEVICE, capacity `dst_capacity` >= block_len(b).
 *   block_start_out  HOST, optional: receives b * 16384.
 *   block_len_out    HOST, optional: receives block_len(b) (16384 except for a short last block). */
int aceapex_seek(aceapex_ctx *ctx, uint64_t coord, void *d_dst, size_t dst_capacity,
                 uint64_t *block_start_out, uint32_t *block_len_out, void *cuda_stream);

/* Synchronises `cuda_stream`, then returns ACEAPEX_OK or ACEAPEX_E_CORRUPT according to the
 * sticky device status word; `first_bad_block` (HOST, optional) receives the lowest block id
 * that raised it (UINT64_MAX if none). `clear` != 0 resets the word. */
int aceapex_device_status(aceapex_ctx *ctx, void *cuda_stream, uint64_t *first_bad_block, int clear);

/* Number of kernels the library has launched on behalf of this context since open (HOST-side
 * counter; used by bench.py's gpu_launches). */
uint64_t aceapex_launch_count(const aceapex_ctx *ctx);

/* Test / profiling hook: entropy-decode the token streams of blocks [first, first+count) into
 * caller memory without running the match layer (the paper's harness checks the entropy layer
 * round trip on its own).
 *   d_lit  DEVICE, count*16384 bytes: block i's LIT stream at i*16384
 *   d_len  DEVICE, count*8192 bytes:  block i's LEN stream at i*8192   (block size / 2)
 *   d_off  DEVICE, count*32768 bytes: block i's OFF stream at i*32768  (2 x block size)
 * count <= n_slots. */
int aceapex_decode_streams(aceapex_ctx *ctx, uint64_t first, size_t count, void *d_lit, void *d_len,
                           void *d_off, void *cuda_stream);

/* Per-kernel device timing (measurement support for bench.py). While
 * enabled, every kernel the library launches is bracketed by two CUDA events on the stream it
 * is launched on. aceapex_profile_read synchronises the device and returns, for each kernel id
 * in [0, ACEAPEX_N_KERNELS), the launches and the summed device milliseconds since the last
 * read (HOST arrays of ACEAPEX_N_KERNELS entries; either may be NULL), then resets the sums. */
enum { ACEAPEX_N_KERNELS = 16 };
int aceapex_profile_enable(aceapex_ctx *ctx, int on);
int aceapex_profile_read(aceapex_ctx *ctx, uint64_t *launches, double *ms);
/* Name of kernel id `id` (NULL if id is not used). */
const char *aceapex_kernel_name(int id);

const char *aceapex_strerror(int code);

void aceapex_close(aceapex_ctx *ctx);

/* aceapex_decode_all_static: aceapex_decode_all for callers that cannot allocate (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc). No context, no caller scratch: the whole decode - both
 * layers of every block, PAPER.md:76 - is enqueued on `cuda_stream` by this one call, which allocates nothing (no
 * cudaMalloc / cudaFree, no host allocation), never synchronises and reads nothing back. The kernels' scratch (control
 * words, done flags, the slots with the decoded token streams) lives in ONE file-scope array in device memory of
 * ACEAPEX_STATIC_SCRATCH_BYTES (8 MiB), which every GPU that loads the library holds until the process exits.
 *   d_container  DEVICE, 16-byte aligned, `nbytes` long; FORMAT.md container.
 *   h_header     HOST, the container's first 64 bytes (required: the call does not read the device).
 *   max_n_seq    upper bound on the sequences per block of this container (aceapex_info.max_n_seq of an earlier
 *                aceapex_open, or what the encoder promised); 0 = the format maximum (block size / 4), which costs
 *                speed and slots. A block with more sequences is left unwritten and reported in d_status.
 *   d_out        DEVICE, capacity `out_capacity` >= total_len; receives out[0, total_len).
 *   d_status     DEVICE, optional, 32 bytes, 8-byte aligned: after the decode the stream copies there
 *                { u64 first_bad_block (~0 = none), u64 blocks_complete, u64 reserved, u32 status (0 = ok, else the
 *                sticky bits of a corrupt container), u32 reserved }.
 * Limits (else ACEAPEX_E_CAPACITY, nothing enqueued): at most ACEAPEX_STATIC_MAX_BLOCKS (4,096) blocks = 64 MiB of
 * output, and the bookkeeping plus at least one slot must fit the array; the blocks are decoded in sub-batches of
 * as many slots as fit (about 230 at max_n_seq 1,000). Other errors: ACEAPEX_E_ARG, ACEAPEX_E_FORMAT
 * (header), ACEAPEX_E_CUDA. The array is shared by ALL calls of a process on that GPU and keeps the last call's
 * contents: every call clears what must start at zero on its stream first, so calls in stream order are
 * independent - but two calls that overlap on the GPU (different streams, or graphs launched concurrently) race
 * on it and corrupt each other. Matches the output of aceapex_decode_all bit for bit. */
enum { ACEAPEX_STATIC_SCRATCH_BYTES = 8 << 20, ACEAPEX_STATIC_MAX_BLOCKS = 4096 };
int aceapex_decode_all_static(const void *d_container, size_t nbytes, const void *h_header, uint32_t max_n_seq,
                              void *d_out, size_t out_capacity, void *d_status, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* ACEAPEX_H */
