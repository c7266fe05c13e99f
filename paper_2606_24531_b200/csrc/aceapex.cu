// C-ABI of include/aceapex.h: host-side header parse, scratch layout, launch sequencing.
// Every step of the decode runs in the kernels of entropy.cuh / match.cuh / seek.cuh; there is
// no CPU decode path in this library.
#include "../../include/aceapex.h"

#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "seek.cuh"

using namespace aceapex;

enum KernelId { K_SCAN = 0, K_ENTROPY, K_MATCH, K_EXPORT, K_SEEK_FUSED, K_COUNT };
static const char *const kKernelNames[K_COUNT] = { "k_scan_records", "k_entropy", "k_match", "k_export_streams", "k_seek_fused" };
static_assert(K_COUNT <= ACEAPEX_N_KERNELS, "kernel id table");

struct ProfRec { int id; cudaEvent_t e0, e1; };

struct aceapex_ctx {
    Container cv{};
    aceapex_info info{};
    SlotLayout sl{};
    Scratch sc{};
    bool have_scratch = false;
    Control *open_ctl = nullptr;          // tiny internal allocation used by the open-time scan
    uint32_t epoch = 0, tag = 0;
    uint64_t launches = 0;
    int sm_count = 0;
    int match_ctas_per_sm = 0;
    int entropy_ctas_per_sm = 0;
    int seek_ctas_per_sm = 0;
    int device = 0;
    bool prof = false;
    std::vector<ProfRec> prof_recs;
    std::vector<cudaEvent_t> prof_pool;
};

// Bracket one kernel launch: counts it and, while profiling, records an event pair around it.
struct LaunchScope {
    aceapex_ctx *c; cudaStream_t st; bool on;
    LaunchScope(aceapex_ctx *c_, int id, cudaStream_t st_) : c(c_), st(st_), on(c_->prof)
    {
        c->launches++;
        if (!on) return;
        ProfRec r; r.id = id;
        for (cudaEvent_t *e : { &r.e0, &r.e1 }) {
            if (!c->prof_pool.empty()) { *e = c->prof_pool.back(); c->prof_pool.pop_back(); }
            else if (cudaEventCreate(e) != cudaSuccess) { on = false; return; }
        }
        cudaEventRecord(r.e0, st);
        c->prof_recs.push_back(r);
    }
    ~LaunchScope() { if (on) cudaEventRecord(c->prof_recs.back().e1, st); }
};

namespace {

inline uint32_t rd32(const uint8_t *p) { return (uint32_t)p[0] | (uint32_t)p[1] << 8 | (uint32_t)p[2] << 16 | (uint32_t)p[3] << 24; }
inline uint64_t rd64(const uint8_t *p) { return (uint64_t)rd32(p) | (uint64_t)rd32(p + 4) << 32; }
inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

struct ScratchOffsets { size_t ctl, done, mark, slot_of, list, ids, slots, pend, total, zero_bytes; };

ScratchOffsets scratch_offsets(uint64_t n_blocks, const SlotLayout &sl, size_t n_slots, size_t n_targets)
{
    ScratchOffsets o;
    size_t p = 0;
    o.ctl = p; p += sizeof(Control);
    o.done = p; p += 4 * (size_t)n_blocks;
    o.mark = p; p += 4 * (size_t)n_blocks;
    p = align_up(p, 8);
    o.slot_of = p; p += 8 * (size_t)n_blocks;
    o.zero_bytes = p;                          // everything up to here is zeroed by set_scratch
    p = align_up(p, 8);
    o.list = p; p += 8 * n_slots;
    o.ids = p; p += 8 * (n_targets ? n_targets : 1);
    p = align_up(p, 256);
    o.slots = p; p += n_slots * (size_t)sl.stride;
    p = align_up(p, 256);
    o.pend = p; p += n_targets * (size_t)kB * 8;
    o.total = align_up(p, 256);
    return o;
}

inline uint32_t block_len_host(const aceapex_ctx *c, uint64_t b)
{
    uint64_t rest = c->info.total_len - (b << kBlockLog2);
    return rest < kB ? (uint32_t)rest : kB;
}

inline size_t entropy_smem() { return kEntropySmem; }
inline size_t match_smem(const aceapex_ctx *c) { return match_smem_bytes(c->sl.ms, c->cv.W); }

// Persistent match kernel: as many CTAs as fit on the device at once (plus nothing: the helper that
// keeps the watermark is one of them), but never more than blocks + 1.
uint32_t match_grid(aceapex_ctx *c, uint32_t count)
{
    if (c->match_ctas_per_sm == 0) {
        int nb = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_match<16>, (int)kMatchThreads, match_smem(c)) != cudaSuccess || nb < 1) nb = 1;
        c->match_ctas_per_sm = nb;
    }
    const uint64_t cap = (uint64_t)c->match_ctas_per_sm * (uint64_t)c->sm_count;
    const uint64_t want = (uint64_t)count + 1;
    return (uint32_t)(want < cap ? want : cap);
}

int launch_entropy(aceapex_ctx *c, const uint64_t *list, const uint32_t *n_list, uint32_t max_slots, uint64_t first,
                   uint32_t count, cudaStream_t st, uint32_t reset_watermark = 0, uint64_t wm_init = 0)
{
    uint32_t units = 3 * (list ? max_slots : count);
    uint32_t grid = (units + kEntropyWarps - 1) / kEntropyWarps;
    if (c->entropy_ctas_per_sm == 0) {         // persistent warps: one wave of resident CTAs (2 of 16 warps per SM)
        int nb = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_entropy, 32 * (int)kEntropyWarps, entropy_smem()) != cudaSuccess || nb < 1) nb = 1;
        c->entropy_ctas_per_sm = nb;
    }
    uint32_t cap = (uint32_t)c->sm_count * (uint32_t)c->entropy_ctas_per_sm;
    if (grid > cap) grid = cap;
    if (grid == 0) return ACEAPEX_OK;
    {
        LaunchScope ls(c, K_ENTROPY, st);
        k_entropy<<<grid, 32 * kEntropyWarps, entropy_smem(), st>>>(c->cv, c->sl, c->sc.slots, list, n_list, max_slots, first, count,
                                                     c->sc.ctl, reset_watermark, (unsigned long long)wm_init);
    }
    return cudaGetLastError() == cudaSuccess ? ACEAPEX_OK : ACEAPEX_E_CUDA;
}

// One group of at most n_targets blocks through the fused isolated-decode kernel. `h_ids` == nullptr: the
// consecutive blocks id0, id0 + 1, ... (range mode when range_lo_blocks > 0: see seek.cuh chase_byte).
int launch_seek_group(aceapex_ctx *c, const uint64_t *h_ids, uint64_t id0, uint32_t nt, uint8_t *d_out, uint64_t out_base,
                      bool absolute, bool range_mode, uint64_t range_lo, cudaStream_t st)
{
    const uint32_t S = (uint32_t)(c->sc.n_slots > 0xFFFFFFFFull / 4 ? 0xFFFFFFFFull / 4 : c->sc.n_slots);
    if (c->seek_ctas_per_sm == 0) {
        int nb = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_seek_fused, 32 * (int)kEntropyWarps, entropy_smem()) != cudaSuccess || nb < 1)
            return ACEAPEX_E_CUDA;
        c->seek_ctas_per_sm = nb;
    }
    const uint32_t kMaxHops = 1u << 16;
    if (c->tag > 0xFFFFFFFFu - 2 * kMaxHops) {                         // hop tags would wrap: start over
        if (cudaMemsetAsync(c->sc.mark, 0, 4 * (size_t)c->cv.n_blocks, st) != cudaSuccess) return ACEAPEX_E_CUDA;
        c->tag = 0;
    }
    SeekArgs a;
    a.pend = c->sc.pend; a.mark = c->sc.mark; a.slot_of = c->sc.slot_of; a.list = c->sc.list;
    a.slots = c->sc.slots; a.out = d_out;
    a.out_base = out_base; a.nt = nt; a.absolute = absolute ? 1u : 0u; a.max_slots = S;
    a.tag0 = c->tag + 1; a.max_hops = kMaxHops;
    a.range_mode = range_mode ? 1u : 0u; a.range_lo = range_lo;
    c->tag += kMaxHops;
    if (!h_ids || nt == 1) {
        a.ids = nullptr; a.one_id = h_ids ? h_ids[0] : id0;            // consecutive targets need no copy at all
    } else {
        if (cudaMemcpyAsync(c->sc.ids, h_ids, 8 * (size_t)nt, cudaMemcpyHostToDevice, st) != cudaSuccess) return ACEAPEX_E_CUDA;
        a.ids = c->sc.ids; a.one_id = 0;
    }
    // all CTAs must be co-resident (grid barrier): one CTA per SM for a few targets (cheaper
    // barriers), the full occupancy for batches
    uint32_t grid = (uint32_t)c->sm_count * (nt <= 4 ? 1u : (uint32_t)c->seek_ctas_per_sm);
    Control *ctl = c->sc.ctl;
    void *params[] = { &c->cv, &c->sl, &a, &ctl };
    {
        LaunchScope ls(c, K_SEEK_FUSED, st);
        if (cudaLaunchCooperativeKernel((const void *)k_seek_fused, dim3(grid), dim3(32 * kEntropyWarps), params, entropy_smem(), st) !=
            cudaSuccess)
            return ACEAPEX_E_CUDA;
    }
    return ACEAPEX_OK;
}

// Blocks [first, first + count) through both layers into d_out (block first + i at d_out + i * 16384), in
// sub-batches of the scratch's slot count (PAPER.md:112 decodes a whole file in sub-batches). first == 0 with
// count == n_blocks is decode_all. For first > 0 (PAPER.md:104 range decode) the sources that lie below the
// range are not in the buffer: before a sub-batch is entropy-decoded and matched, the fused isolated kernel
// follows exactly those bytes to their origins through the compressed data and writes them in place; the match
// kernel then takes every other byte from the range's own buffer.
int decode_span(aceapex_ctx *c, uint64_t first, uint64_t count, uint8_t *d_out, cudaStream_t st)
{
    if (++c->epoch == 0) {   // epoch wrapped: stale done flags could alias
        if (cudaMemsetAsync(c->sc.done, 0, 4 * (size_t)c->cv.n_blocks, st) != cudaSuccess) return ACEAPEX_E_CUDA;
        c->epoch = 1;
    }
    const uint32_t align = ((uintptr_t)d_out & 15) == 0 ? 16u : (((uintptr_t)d_out & 3) == 0 ? 4u : 1u);
    const uint64_t range_lo = first << kBlockLog2;
    uint8_t *out_virtual = d_out - range_lo;                           // absolute output offset -> address
    uint64_t step = c->sc.n_slots;
    if (first > 0 && c->sc.n_targets < step) step = c->sc.n_targets;
    for (uint64_t f = first; f < first + count; f += step) {
        const uint64_t rest = first + count - f;
        const uint32_t cnt = (uint32_t)(rest < step ? rest : step);
        if (first > 0) {
            int rc = launch_seek_group(c, nullptr, f, cnt, d_out, f - first, false, true, range_lo, st);
            if (rc != ACEAPEX_OK) return rc;
        }
        // the first entropy launch of the call also re-arms the watermark (nothing reads it before the match kernel)
        int rc = launch_entropy(c, nullptr, nullptr, 0, f, cnt, st, f == first ? 1u : 0u, first);
        if (rc != ACEAPEX_OK) return rc;
        {
            LaunchScope ls(c, K_MATCH, st);
            const uint32_t grid = match_grid(c, cnt);
            if (align >= 16) k_match<16><<<grid, kMatchThreads, match_smem(c), st>>>(c->cv, c->sl, c->sc.slots, f, cnt, out_virtual,
                                                                    c->sc.ctl, c->sc.done, c->epoch, range_lo);
            else if (align >= 4) k_match<4><<<grid, kMatchThreads, match_smem(c), st>>>(c->cv, c->sl, c->sc.slots, f, cnt, out_virtual,
                                                                    c->sc.ctl, c->sc.done, c->epoch, range_lo);
            else k_match<1><<<grid, kMatchThreads, match_smem(c), st>>>(c->cv, c->sl, c->sc.slots, f, cnt, out_virtual,
                                                                    c->sc.ctl, c->sc.done, c->epoch, range_lo);
        }
        if (cudaGetLastError() != cudaSuccess) return ACEAPEX_E_CUDA;
    }
    return ACEAPEX_OK;
}

}  // namespace

extern "C" {

int aceapex_version(void) { return 100; }

const char *aceapex_strerror(int code)
{
    switch (code) {
    case ACEAPEX_OK: return "ok";
    case ACEAPEX_E_ARG: return "bad argument";
    case ACEAPEX_E_FORMAT: return "bad container header";
    case ACEAPEX_E_CAPACITY: return "buffer too small";
    case ACEAPEX_E_CORRUPT: return "corrupt container";
    case ACEAPEX_E_RANGE: return "block id or coordinate out of range";
    case ACEAPEX_E_NOMEM: return "out of host memory";
    case ACEAPEX_E_CUDA: return "CUDA runtime error";
    case ACEAPEX_E_STATE: return "scratch not set";
    default: return "unknown error";
    }
}

int aceapex_open(const void *d_container, size_t nbytes, const void *h_header, aceapex_ctx **out)
{
    if (!d_container || !out) return ACEAPEX_E_ARG;
    *out = nullptr;
    if ((uintptr_t)d_container & 15) return ACEAPEX_E_ARG;
    if (nbytes < kHeaderBytes) return ACEAPEX_E_FORMAT;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return ACEAPEX_E_CUDA;
    uint8_t h[kHeaderBytes];
    if (h_header) memcpy(h, h_header, kHeaderBytes);
    else if (cudaMemcpy(h, d_container, kHeaderBytes, cudaMemcpyDeviceToHost) != cudaSuccess) return ACEAPEX_E_CUDA;

    // FORMAT.md section 1
    if (memcmp(h, "ACEAPEX1", 8) != 0 || rd32(h + 8) != 1) return ACEAPEX_E_FORMAT;
    if (h[12] != kBlockLog2 || (h[13] != 4 && h[13] != 8) || h[14] != kLanes || h[15] != kProbBits) return ACEAPEX_E_FORMAT;
    const uint64_t total_len = rd64(h + 16), n_blocks = rd64(h + 24);
    const uint32_t D = rd32(h + 32), R = rd32(h + 36), max_level = rd32(h + 40);
    const uint64_t index_off = rd64(h + 48), payload_off = rd64(h + 56);
    if (n_blocks != (total_len + kB - 1) / kB || n_blocks > (1ull << 32) - 2) return ACEAPEX_E_FORMAT;
    if (index_off != kHeaderBytes || max_level > 15) return ACEAPEX_E_FORMAT;
    const uint64_t index_bytes = (n_blocks + 1) * 8 + n_blocks * 3 * kLanes * 4;
    if (payload_off != ((kHeaderBytes + index_bytes + 15) & ~15ull) || payload_off > nbytes) return ACEAPEX_E_FORMAT;

    aceapex_ctx *c = new (std::nothrow) aceapex_ctx();
    if (!c) return ACEAPEX_E_NOMEM;
    c->device = dev;
    const uint8_t *base = static_cast<const uint8_t *>(d_container);
    c->cv.base = base;
    c->cv.rec_off = reinterpret_cast<const uint64_t *>(base + kHeaderBytes);
    c->cv.states = reinterpret_cast<const uint32_t *>(base + kHeaderBytes + (n_blocks + 1) * 8);
    c->cv.payload = base + payload_off;
    c->cv.total_len = total_len;
    c->cv.n_blocks = n_blocks;
    c->cv.W = h[13]; c->cv.D = D; c->cv.R = R; c->cv.max_level = max_level;
    c->epoch = 0; c->tag = 0;

    int rc = ACEAPEX_OK;
    uint64_t edge[2] = { 0, 0 };   // rec_off[0], rec_off[n_blocks]
    if (cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) rc = ACEAPEX_E_CUDA;
    if (rc == ACEAPEX_OK && cudaMemcpy(&edge[0], c->cv.rec_off, 8, cudaMemcpyDeviceToHost) != cudaSuccess) rc = ACEAPEX_E_CUDA;
    if (rc == ACEAPEX_OK && cudaMemcpy(&edge[1], c->cv.rec_off + n_blocks, 8, cudaMemcpyDeviceToHost) != cudaSuccess) rc = ACEAPEX_E_CUDA;
    if (rc == ACEAPEX_OK && (edge[0] != 0 || payload_off + edge[1] > nbytes)) rc = ACEAPEX_E_FORMAT;
    c->cv.payload_bytes = edge[1];

    if (rc == ACEAPEX_OK && cudaMalloc(&c->open_ctl, sizeof(Control)) != cudaSuccess) rc = ACEAPEX_E_CUDA;
    if (rc == ACEAPEX_OK) {
        Control init;
        memset(&init, 0, sizeof init);
        init.first_bad = ~0ull;
        if (cudaMemcpy(c->open_ctl, &init, sizeof init, cudaMemcpyHostToDevice) != cudaSuccess) rc = ACEAPEX_E_CUDA;
    }
    if (rc == ACEAPEX_OK && n_blocks) {
        // one pass over all record headers (one entropy entry point per block)
        const uint32_t grid = (uint32_t)((n_blocks + 255) / 256);
        k_scan_records<<<grid, 256>>>(c->cv, c->open_ctl);
        c->launches++;
        if (cudaGetLastError() != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) rc = ACEAPEX_E_CUDA;
    }
    Control res;
    memset(&res, 0, sizeof res);
    if (rc == ACEAPEX_OK && cudaMemcpy(&res, c->open_ctl, sizeof res, cudaMemcpyDeviceToHost) != cudaSuccess) rc = ACEAPEX_E_CUDA;
    if (rc == ACEAPEX_OK && res.status) rc = ACEAPEX_E_CORRUPT;
    if (rc == ACEAPEX_OK) {
        if (cudaFuncSetAttribute(k_entropy, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)entropy_smem()) != cudaSuccess ||
            cudaFuncSetAttribute(k_seek_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)entropy_smem()) != cudaSuccess)
            rc = ACEAPEX_E_CUDA;
    }
    if (rc != ACEAPEX_OK) { aceapex_close(c); return rc; }

    c->sl = make_slot_layout(res.max_n_seq, c->cv.W);
    // The attribute belongs to the function, not to this context: set it to the format maximum (block size / 4
    // sequences, 8-byte offsets), or to what the device offers if that is less (32 KiB blocks), so that contexts of
    // different containers cannot lower each other's limit. A container whose densest block needs more than the
    // device has cannot be decoded by this build.
    {
        int optin = 0;
        if (cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) { aceapex_close(c); return ACEAPEX_E_CUDA; }
        const size_t avail = (size_t)optin > 2048 ? (size_t)optin - 2048 : 0;   // the kernel's static shared memory
        const size_t fmt_max = match_smem_bytes(kMaxSeq, 8);
        if (match_smem(c) > avail) { aceapex_close(c); return ACEAPEX_E_CAPACITY; }
        if (cudaFuncSetAttribute(k_match<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(fmt_max < avail ? fmt_max : avail)) != cudaSuccess ||
            cudaFuncSetAttribute(k_match<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(fmt_max < avail ? fmt_max : avail)) != cudaSuccess ||
            cudaFuncSetAttribute(k_match<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(fmt_max < avail ? fmt_max : avail)) != cudaSuccess) {
            aceapex_close(c);
            return ACEAPEX_E_CUDA;
        }
    }
    c->info.total_len = total_len;
    c->info.n_blocks = n_blocks;
    c->info.container_bytes = payload_off + edge[1];
    c->info.block_size = kB;
    c->info.offset_width = c->cv.W;
    c->info.max_depth = D;
    c->info.window = R;
    c->info.max_level = max_level;
    c->info.max_n_seq = res.max_n_seq;
    *out = c;
    return ACEAPEX_OK;
}

void aceapex_close(aceapex_ctx *c)
{
    if (!c) return;
    if (c->open_ctl) cudaFree(c->open_ctl);
    for (ProfRec &r : c->prof_recs) { cudaEventDestroy(r.e0); cudaEventDestroy(r.e1); }
    for (cudaEvent_t e : c->prof_pool) cudaEventDestroy(e);
    delete c;
}

int aceapex_info_get(const aceapex_ctx *c, aceapex_info *out)
{
    if (!c || !out) return ACEAPEX_E_ARG;
    *out = c->info;
    return ACEAPEX_OK;
}

size_t aceapex_scratch_bytes(const aceapex_ctx *c, size_t n_slots, size_t n_targets)
{
    if (!c || n_slots == 0) return 0;
    return scratch_offsets(c->cv.n_blocks, c->sl, n_slots, n_targets).total;
}

int aceapex_set_scratch(aceapex_ctx *c, void *d_scratch, size_t nbytes, size_t n_slots, size_t n_targets,
                        void *cuda_stream)
{
    if (!c || !d_scratch || n_slots == 0 || n_slots > 0xFFFFFFFFull / 3 || n_targets > (1u << 18)) return ACEAPEX_E_ARG;
    if ((uintptr_t)d_scratch & 255) return ACEAPEX_E_ARG;
    const ScratchOffsets o = scratch_offsets(c->cv.n_blocks, c->sl, n_slots, n_targets);
    if (nbytes < o.total) return ACEAPEX_E_CAPACITY;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    uint8_t *p = static_cast<uint8_t *>(d_scratch);
    c->sc.ctl = reinterpret_cast<Control *>(p + o.ctl);
    c->sc.done = reinterpret_cast<uint32_t *>(p + o.done);
    c->sc.mark = reinterpret_cast<uint32_t *>(p + o.mark);
    c->sc.slot_of = reinterpret_cast<unsigned long long *>(p + o.slot_of);
    c->sc.list = reinterpret_cast<uint64_t *>(p + o.list);
    c->sc.ids = reinterpret_cast<uint64_t *>(p + o.ids);
    c->sc.slots = p + o.slots;
    c->sc.pend = reinterpret_cast<uint64_t *>(p + o.pend);
    c->sc.n_slots = n_slots;
    c->sc.n_targets = n_targets;
    c->epoch = 0;
    c->tag = 0;
    if (cudaMemsetAsync(p, 0, o.zero_bytes, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    if (cudaMemsetAsync(&c->sc.ctl->first_bad, 0xFF, 8, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    c->have_scratch = true;
    return ACEAPEX_OK;
}

int aceapex_decode_all(aceapex_ctx *c, void *d_out, size_t out_capacity, void *cuda_stream)
{
    if (!c || (!d_out && c->info.total_len)) return ACEAPEX_E_ARG;
    if (!c->have_scratch) return ACEAPEX_E_STATE;
    if (out_capacity < c->info.total_len) return ACEAPEX_E_CAPACITY;
    if (c->cv.n_blocks == 0) return ACEAPEX_OK;
    return decode_span(c, 0, c->cv.n_blocks, static_cast<uint8_t *>(d_out), static_cast<cudaStream_t>(cuda_stream));
}

int aceapex_decode_range(aceapex_ctx *c, uint64_t first, uint64_t count, void *d_out, size_t out_capacity, void *cuda_stream)
{
    if (!c || (count && !d_out)) return ACEAPEX_E_ARG;
    if (first + count < first || first + count > c->cv.n_blocks) return ACEAPEX_E_RANGE;
    if (count == 0) return ACEAPEX_OK;
    if (!c->have_scratch || (first > 0 && c->sc.n_targets == 0)) return ACEAPEX_E_STATE;
    const uint64_t last = first + count - 1;
    const size_t need = (size_t)((count - 1) << kBlockLog2) + block_len_host(c, last);
    if (out_capacity < need) return ACEAPEX_E_CAPACITY;
    return decode_span(c, first, count, static_cast<uint8_t *>(d_out), static_cast<cudaStream_t>(cuda_stream));
}

int aceapex_decode_streams(aceapex_ctx *c, uint64_t first, size_t count, void *d_lit, void *d_len, void *d_off,
                           void *cuda_stream)
{
    if (!c || !d_lit || !d_len || !d_off) return ACEAPEX_E_ARG;
    if (!c->have_scratch) return ACEAPEX_E_STATE;
    if (count > c->sc.n_slots) return ACEAPEX_E_CAPACITY;
    if (first + count > c->cv.n_blocks || first + count < first) return ACEAPEX_E_RANGE;
    if (count == 0) return ACEAPEX_OK;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    int rc = launch_entropy(c, nullptr, nullptr, 0, first, (uint32_t)count, st);
    if (rc != ACEAPEX_OK) return rc;
    {
        LaunchScope ls(c, K_EXPORT, st);
        k_export_streams<<<(uint32_t)count, 256, 0, st>>>(c->cv, c->sl, c->sc.slots, first, (uint32_t)count,
                                                          static_cast<uint8_t *>(d_lit), static_cast<uint8_t *>(d_len),
                                                          static_cast<uint8_t *>(d_off));
    }
    return cudaGetLastError() == cudaSuccess ? ACEAPEX_OK : ACEAPEX_E_CUDA;
}

int aceapex_decode_blocks(aceapex_ctx *c, const uint64_t *h_ids, size_t n_ids, void *d_out, size_t out_capacity,
                          uint32_t flags, void *cuda_stream)
{
    if (!c || (n_ids && (!h_ids || !d_out)) || flags > ACEAPEX_ABSOLUTE) return ACEAPEX_E_ARG;
    if (n_ids == 0) return ACEAPEX_OK;
    if (!c->have_scratch || c->sc.n_targets == 0) return ACEAPEX_E_STATE;
    const bool absolute = flags == ACEAPEX_ABSOLUTE;
    size_t need = 0;
    for (size_t i = 0; i < n_ids; i++) {
        if (h_ids[i] >= c->cv.n_blocks) return ACEAPEX_E_RANGE;
        const size_t end = ((absolute ? (size_t)h_ids[i] : i) << kBlockLog2) + block_len_host(c, h_ids[i]);
        if (end > need) need = end;
    }
    if (out_capacity < need) return ACEAPEX_E_CAPACITY;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    for (size_t base = 0; base < n_ids; base += c->sc.n_targets) {
        const uint32_t nt = (uint32_t)(n_ids - base < c->sc.n_targets ? n_ids - base : c->sc.n_targets);
        int rc = launch_seek_group(c, h_ids + base, 0, nt, static_cast<uint8_t *>(d_out), (uint64_t)base, absolute, false, 0, st);
        if (rc != ACEAPEX_OK) return rc;
    }
    return cudaGetLastError() == cudaSuccess ? ACEAPEX_OK : ACEAPEX_E_CUDA;
}

int aceapex_seek(aceapex_ctx *c, uint64_t coord, void *d_dst, size_t dst_capacity, uint64_t *block_start_out,
                 uint32_t *block_len_out, void *cuda_stream)
{
    if (!c || !d_dst) return ACEAPEX_E_ARG;
    if (coord >= c->info.total_len) return ACEAPEX_E_RANGE;
    const uint64_t b = coord >> kBlockLog2;          // the single coordinate
    const uint32_t len = block_len_host(c, b);
    if (dst_capacity < len) return ACEAPEX_E_CAPACITY;
    if (block_start_out) *block_start_out = b << kBlockLog2;
    if (block_len_out) *block_len_out = len;
    return aceapex_decode_blocks(c, &b, 1, d_dst, dst_capacity, ACEAPEX_PACKED, cuda_stream);
}

int aceapex_device_status(aceapex_ctx *c, void *cuda_stream, uint64_t *first_bad_block, int clear)
{
    if (!c) return ACEAPEX_E_ARG;
    if (!c->have_scratch) return ACEAPEX_E_STATE;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    Control h;
    if (cudaMemcpyAsync(&h, c->sc.ctl, sizeof h, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return ACEAPEX_E_CUDA;
    if (first_bad_block) *first_bad_block = h.first_bad;
    if (clear && h.status) {
        if (cudaMemsetAsync(&c->sc.ctl->status, 0, 4, st) != cudaSuccess) return ACEAPEX_E_CUDA;
        if (cudaMemsetAsync(&c->sc.ctl->first_bad, 0xFF, 8, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    }
    return h.status ? ACEAPEX_E_CORRUPT : ACEAPEX_OK;
}

uint64_t aceapex_launch_count(const aceapex_ctx *c) { return c ? c->launches : 0; }

int aceapex_profile_enable(aceapex_ctx *c, int on)
{
    if (!c) return ACEAPEX_E_ARG;
    c->prof = on != 0;
    return ACEAPEX_OK;
}

int aceapex_profile_read(aceapex_ctx *c, uint64_t *launches, double *ms)
{
    if (!c) return ACEAPEX_E_ARG;
    if (cudaDeviceSynchronize() != cudaSuccess) return ACEAPEX_E_CUDA;
    for (int i = 0; i < ACEAPEX_N_KERNELS; i++) {
        if (launches) launches[i] = 0;
        if (ms) ms[i] = 0.0;
    }
    int rc = ACEAPEX_OK;
    for (ProfRec &r : c->prof_recs) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, r.e0, r.e1) != cudaSuccess) rc = ACEAPEX_E_CUDA;
        if (launches) launches[r.id]++;
        if (ms) ms[r.id] += (double)t;
        c->prof_pool.push_back(r.e0);
        c->prof_pool.push_back(r.e1);
    }
    c->prof_recs.clear();
    return rc;
}

const char *aceapex_kernel_name(int id) { return id >= 0 && id < K_COUNT ? kKernelNames[id] : nullptr; }

// ---- aceapex_decode_all_static: decode_all without any allocation ------------------------------------------------
//
// The scratch of the two decode_all kernels in a file-scope device array instead of caller memory. In host code the
// array's NAME is a host-side stand-in, not a device address (a kernel handed it would fault or use the wrong
// memory): its address on the current device comes from cudaGetSymbolAddress, once per device.
static __device__ __align__(256) unsigned char g_static_scratch[ACEAPEX_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kMaxStaticDevices = 64;
struct StaticDevice { bool ready; uint8_t *scratch; int sm_count; size_t smem_avail; };
StaticDevice g_static_dev[kMaxStaticDevices];
std::mutex g_static_mutex;

// Set-up, once per device, with that device current: the array's device address, the kernels' shared-memory
// attributes, the SM count. No allocation.
int static_device(int dev, StaticDevice *out)
{
    if (dev < 0 || dev >= kMaxStaticDevices) return ACEAPEX_E_ARG;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice &d = g_static_dev[dev];
    if (!d.ready) {
        void *ptr = nullptr;
        if (cudaGetSymbolAddress(&ptr, g_static_scratch) != cudaSuccess || !ptr) return ACEAPEX_E_CUDA;
        int optin = 0;
        if (cudaDeviceGetAttribute(&d.sm_count, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess)
            return ACEAPEX_E_CUDA;
        d.smem_avail = (size_t)optin > 2048 ? (size_t)optin - 2048 : 0;
        const size_t fmt_max = match_smem_bytes(kMaxSeq, 8);
        const int msm = (int)(fmt_max < d.smem_avail ? fmt_max : d.smem_avail);
        if (cudaFuncSetAttribute(k_entropy, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)entropy_smem()) != cudaSuccess ||
            cudaFuncSetAttribute(k_match<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, msm) != cudaSuccess ||
            cudaFuncSetAttribute(k_match<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, msm) != cudaSuccess ||
            cudaFuncSetAttribute(k_match<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, msm) != cudaSuccess)
            return ACEAPEX_E_CUDA;
        d.scratch = static_cast<uint8_t *>(ptr);
        d.ready = true;
    }
    *out = d;
    return ACEAPEX_OK;
}

}  // namespace

int aceapex_decode_all_static(const void *d_container, size_t nbytes, const void *h_header, uint32_t max_n_seq,
                              void *d_out, size_t out_capacity, void *d_status, void *cuda_stream)
{
    if (!d_container || !h_header || ((uintptr_t)d_container & 15) || ((uintptr_t)d_status & 7)) return ACEAPEX_E_ARG;
    if (nbytes < kHeaderBytes) return ACEAPEX_E_FORMAT;
    const uint8_t *h = static_cast<const uint8_t *>(h_header);
    // FORMAT.md section 1 (the same checks as aceapex_open, from the caller's host copy of the header)
    if (memcmp(h, "ACEAPEX1", 8) != 0 || rd32(h + 8) != 1) return ACEAPEX_E_FORMAT;
    if (h[12] != kBlockLog2 || (h[13] != 4 && h[13] != 8) || h[14] != kLanes || h[15] != kProbBits) return ACEAPEX_E_FORMAT;
    const uint64_t total_len = rd64(h + 16), n_blocks = rd64(h + 24);
    const uint64_t index_off = rd64(h + 48), payload_off = rd64(h + 56);
    if (n_blocks != (total_len + kB - 1) / kB || n_blocks > (1ull << 32) - 2) return ACEAPEX_E_FORMAT;
    if (index_off != kHeaderBytes || rd32(h + 40) > 15) return ACEAPEX_E_FORMAT;
    const uint64_t index_bytes = (n_blocks + 1) * 8 + n_blocks * 3 * kLanes * 4;
    if (payload_off != ((kHeaderBytes + index_bytes + 15) & ~15ull) || payload_off > nbytes) return ACEAPEX_E_FORMAT;
    if (!d_out && total_len) return ACEAPEX_E_ARG;
    if (out_capacity < total_len) return ACEAPEX_E_CAPACITY;
    if (n_blocks > ACEAPEX_STATIC_MAX_BLOCKS) return ACEAPEX_E_CAPACITY;
    if (max_n_seq == 0 || max_n_seq > kMaxSeq) max_n_seq = kMaxSeq;

    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return ACEAPEX_E_CUDA;
    StaticDevice sd;
    int rc = static_device(dev, &sd);
    if (rc != ACEAPEX_OK) return rc;
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);

    // a context on the stack (nothing in it allocates), its scratch carved out of the static array
    aceapex_ctx c;
    const uint8_t *base = static_cast<const uint8_t *>(d_container);
    c.cv.base = base;
    c.cv.rec_off = reinterpret_cast<const uint64_t *>(base + kHeaderBytes);
    c.cv.states = reinterpret_cast<const uint32_t *>(base + kHeaderBytes + (n_blocks + 1) * 8);
    c.cv.payload = base + payload_off;
    c.cv.total_len = total_len;
    c.cv.n_blocks = n_blocks;
    c.cv.payload_bytes = nbytes - payload_off;         // upper bound: every record must end inside the caller's buffer
    c.cv.W = h[13]; c.cv.D = rd32(h + 32); c.cv.R = rd32(h + 36); c.cv.max_level = rd32(h + 40);
    c.device = dev;
    c.sm_count = sd.sm_count;
    c.sl = make_slot_layout(max_n_seq, c.cv.W);
    if (match_smem(&c) > sd.smem_avail) return ACEAPEX_E_CAPACITY;
    if (n_blocks == 0) {
        if (d_status && cudaMemsetAsync(d_status, 0, 32, st) != cudaSuccess) return ACEAPEX_E_CUDA;
        if (d_status && cudaMemsetAsync(d_status, 0xFF, 8, st) != cudaSuccess) return ACEAPEX_E_CUDA;
        return ACEAPEX_OK;
    }
    // as many slots as fit the array beside the bookkeeping (at most one per block)
    const ScratchOffsets o1 = scratch_offsets(n_blocks, c.sl, 1, 0);
    if (o1.total > ACEAPEX_STATIC_SCRATCH_BYTES) return ACEAPEX_E_CAPACITY;
    size_t n_slots = 1 + (ACEAPEX_STATIC_SCRATCH_BYTES - o1.total) / ((size_t)c.sl.stride + 8);
    if (n_slots > n_blocks) n_slots = (size_t)n_blocks;
    while (n_slots > 1 && scratch_offsets(n_blocks, c.sl, n_slots, 0).total > ACEAPEX_STATIC_SCRATCH_BYTES) n_slots--;
    const ScratchOffsets o = scratch_offsets(n_blocks, c.sl, n_slots, 0);
    uint8_t *p = sd.scratch;
    c.sc.ctl = reinterpret_cast<Control *>(p + o.ctl);
    c.sc.done = reinterpret_cast<uint32_t *>(p + o.done);
    c.sc.mark = reinterpret_cast<uint32_t *>(p + o.mark);
    c.sc.slot_of = reinterpret_cast<unsigned long long *>(p + o.slot_of);
    c.sc.list = reinterpret_cast<uint64_t *>(p + o.list);
    c.sc.ids = reinterpret_cast<uint64_t *>(p + o.ids);
    c.sc.slots = p + o.slots;
    c.sc.pend = reinterpret_cast<uint64_t *>(p + o.pend);
    c.sc.n_slots = n_slots;
    c.sc.n_targets = 0;
    c.have_scratch = true;
    // The array keeps the previous call's contents: the control words (status, counters) and the done flags must
    // start at zero, first_bad at ~0. (The slots are fully rewritten by the entropy kernel before they are read.)
    if (cudaMemsetAsync(p, 0, o.mark, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    if (cudaMemsetAsync(&c.sc.ctl->first_bad, 0xFF, 8, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    rc = decode_span(&c, 0, n_blocks, static_cast<uint8_t *>(d_out), st);
    if (rc != ACEAPEX_OK) return rc;
    if (d_status && cudaMemcpyAsync(d_status, c.sc.ctl, 32, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    return ACEAPEX_OK;
}

}  // extern "C"
