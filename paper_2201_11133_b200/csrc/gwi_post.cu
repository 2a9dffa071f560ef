// gwi_post.cu -- ensemble mean + strict threshold + run-length trigger clustering (gwi_ensemble_triggers).
//
// Definition (DESIGN.md C.1 "Triggers", readings A18-A22; "height" and "width >= 0.5 s"):
//   pbar[t] = (((p0[t]+p1[t])+p2[t])+...)/(float)M   fixed fp32 expression (tier T1: bit-reproducible)
//   a[t]    = pbar[t] > theta                        strict
//   every maximal run [s,e) of a = 1 with e - s >= L_min is a trigger, sorted by s; runs are carried across
//   consecutive chunks through the caller's carry block and closed at the stream end when last_chunk != 0.
//
// Kernels:
//   k_mask      HBM-bound pass: reads M x N floats once, writes N/8 bytes of bit mask (+ optional pbar).  This is
//               the roofline kernel of the post-processing: 4*M (+4) algorithmic bytes per sample.
//   k_blkflags  per 256-word block "all ones" flag so that long runs are walked 8192 samples per step
//   k_head_run  closes / continues the run carried in from the previous chunk
//   k_runs<0>   one thread per 32-sample word: finds run starts, walks to the run end, counts qualifying runs
//   k_scan      exclusive scan of the per-CTA counts -> output offsets, total -> *d_count
//   k_runs<1>   same walk, writes {slide,start,end} at its slot (records come out sorted by start)
//   k_stats     one CTA per record: peak / mean / model_mask over the run; last CTA updates the carry block
#include <type_traits>

#include "gwi_internal.h"

namespace {

constexpr int WB = 256;    // words per all-ones block
constexpr int RT = 1024;   // threads (= words) per CTA in k_runs
constexpr int ST_THREADS = 1024;   // threads per CTA in k_stats

struct Ptrs {
    const float* p[GWI_MAX_MODELS];
};

struct Carry {             // the caller's opaque carry block (gwi_carry_bytes())
    int32_t open;
    int32_t mask;
    int64_t start;         // global start of the open run
    double sum;
    float peak;
    int32_t pad;
};

struct Header {            // per-call scratch header at the start of the workspace
    Carry in;              // copy of the incoming carry (zero if none)
    int32_t head_emit;     // the carried run closes in this chunk and qualifies -> record 0
    int32_t head_closed;   // the carried run closes in this chunk
    int64_t head_end;      // local index where it closes
    int32_t out_open;      // a run is open at the end of this chunk
    int32_t pad;
    int64_t out_start;     // its global start
    int32_t total;         // records in the output buffer after this call (base + this call's)
    int32_t base;          // records already in the buffer before this call (append mode; else 0)
};

__device__ __forceinline__ float ens_mean(const Ptrs& P, int M, int64_t i)
{
    float s = P.p[0][i];
    for (int j = 1; j < M; j++) s = __fadd_rn(s, P.p[j][i]);
    return __fdiv_rn(s, (float)M);
}

template <bool VEC>
__global__ void k_mask(Ptrs P, int M, int64_t N, float theta, uint32_t* __restrict__ bits, int64_t NW,
                       float* __restrict__ pbar)
{
    const int lane = threadIdx.x & 31;
    const int64_t warp = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int64_t nwarps = ((int64_t)gridDim.x * blockDim.x) >> 5;
    const float fM = (float)M;
    for (int64_t base = warp * 128; base < NW * 32; base += nwarps * 128) {
        int64_t i = base + 4 * lane;
        float m4[4] = {0.f, 0.f, 0.f, 0.f};
        uint32_t nib = 0;
        if (VEC && i + 3 < N) {
            float4 s = *reinterpret_cast<const float4*>(P.p[0] + i);
            for (int j = 1; j < M; j++) {
                float4 v = *reinterpret_cast<const float4*>(P.p[j] + i);
                s.x = __fadd_rn(s.x, v.x), s.y = __fadd_rn(s.y, v.y), s.z = __fadd_rn(s.z, v.z), s.w = __fadd_rn(s.w, v.w);
            }
            m4[0] = __fdiv_rn(s.x, fM), m4[1] = __fdiv_rn(s.y, fM), m4[2] = __fdiv_rn(s.z, fM), m4[3] = __fdiv_rn(s.w, fM);
            nib = (m4[0] > theta) | ((m4[1] > theta) << 1) | ((m4[2] > theta) << 2) | ((m4[3] > theta) << 3);
            if (pbar) *reinterpret_cast<float4*>(pbar + i) = make_float4(m4[0], m4[1], m4[2], m4[3]);
        } else {
            for (int e = 0; e < 4; e++)
                if (i + e < N) {
                    float v = ens_mean(P, M, i + e);
                    nib |= (uint32_t)(v > theta) << e;
                    if (pbar) pbar[i + e] = v;
                }
        }
        uint32_t w = nib << (4 * (lane & 7));
        w |= __shfl_xor_sync(0xffffffffu, w, 1);
        w |= __shfl_xor_sync(0xffffffffu, w, 2);
        w |= __shfl_xor_sync(0xffffffffu, w, 4);
        int64_t wi = (base >> 5) + (lane >> 3);
        if ((lane & 7) == 0 && wi < NW) bits[wi] = w;
    }
}

// Several slides in one launch (the fused slide heads leave one mask per slide, gwi_post_run_bits_batch): slide y works on
// the mask at bits + y * bits_stride, the mean / model bytes at + y * row_stride, its own scratch block (header, flags,
// counts, offsets: ws_stride bytes apart) and its own carry.  A single slide has all strides 0.
struct Batch {
    int64_t bits_stride, row_stride;
    size_t ws_stride;
};
template <class T>
__device__ __forceinline__ T* ws_of(T* p, const Batch& b, int y) { return reinterpret_cast<T*>(reinterpret_cast<char*>(const_cast<typename std::remove_const<T>::type*>(p)) + (size_t)y * b.ws_stride); }

__global__ void k_blkflags(const uint32_t* __restrict__ bits, int64_t NW, uint8_t* __restrict__ flags, Batch bt)
{
    bits += blockIdx.y * bt.bits_stride, flags = ws_of(flags, bt, blockIdx.y);
    int64_t i = (int64_t)blockIdx.x * WB + threadIdx.x;
    int ok = (i < NW) ? (bits[i] == 0xffffffffu) : 0;
    int all = __syncthreads_and(ok);
    if (threadIdx.x == 0) flags[blockIdx.x] = (uint8_t)all;
}

// first index >= pos whose bit is 0 (bits past N are 0), capped at N
__device__ int64_t find_end(const uint32_t* __restrict__ bits, const uint8_t* __restrict__ flags, int64_t NW,
                            int64_t N, int64_t pos)
{
    int64_t i = pos >> 5;
    uint32_t w = ~bits[i] & (0xffffffffu << (pos & 31));
    if (w) return min((int64_t)(i * 32 + __ffs(w) - 1), N);
    i++;
    while (i < NW) {
        if ((i % WB) == 0) {
            while (i + WB <= NW && flags[i / WB]) i += WB;
            if (i >= NW) break;
        }
        // the words up to the next block boundary, eight independent loads at a time (a 1 s run is 128 words: walked one
        // dependent load after the other it was the longest chain of the whole call)
        const int64_t stop = min(NW, (i / WB + 1) * WB);
        for (; i < stop; i += 8) {
            uint32_t v[8];
#pragma unroll
            for (int u = 0; u < 8; u++) v[u] = (i + u < stop) ? ~bits[i + u] : 0u;
#pragma unroll
            for (int u = 0; u < 8; u++)
                if (v[u]) return min((int64_t)((i + u) * 32 + __ffs(v[u]) - 1), N);
        }
        i = stop;
    }
    return N;
}

// shard_begin / shard_end (time-shard mode of the stream driver; -1 = off): global index of the shard's
// first sample / one past its last.  A run that touches either is emitted whatever its length (it may continue in the
// neighbouring shard; the host merges and applies L_min afterwards) and is flagged in model_mask by k_stats.
__global__ void k_head_run(const uint32_t* __restrict__ bits, const uint8_t* __restrict__ flags, int64_t NW, int64_t N,
                           int64_t t0, int64_t Lmin, int last_chunk, const Carry* __restrict__ carry, Header* hd,
                           int64_t shard_begin, int64_t shard_end, Batch bt)
{
    if (threadIdx.x != 0) return;
    bits += blockIdx.x * bt.bits_stride, flags = ws_of(flags, bt, blockIdx.x), hd = ws_of(hd, bt, blockIdx.x);
    if (carry) carry += blockIdx.x;
    Carry c;
    if (carry) c = *carry;
    else { c.open = 0, c.mask = 0, c.start = 0, c.sum = 0.0, c.peak = 0.f, c.pad = 0; }
    hd->in = c;
    hd->head_emit = 0, hd->head_closed = 0, hd->head_end = 0, hd->out_open = 0, hd->out_start = 0, hd->total = 0;
    if (c.open) {
        int64_t e0 = (bits[0] & 1u) ? find_end(bits, flags, NW, N, 0) : 0;
        if (e0 < N || last_chunk) {
            hd->head_closed = 1;
            hd->head_end = e0;
            hd->head_emit = (t0 + e0 - c.start >= Lmin || c.start == shard_begin || t0 + e0 == shard_end) ? 1 : 0;
        } else {
            hd->out_open = 1;
            hd->out_start = c.start;
        }
    }
}

// MODE 0: count qualifying closed runs per CTA.  MODE 1: write the records.
template <int MODE>
__global__ void k_runs(const uint32_t* __restrict__ bits, const uint8_t* __restrict__ flags, int64_t NW, int64_t N,
                       int64_t t0, int64_t Lmin, int last_chunk, int slide, Header* hd, uint32_t* __restrict__ blkcnt,
                       const uint32_t* __restrict__ blkoff, gwi_trigger* __restrict__ out, int capacity,
                       int64_t shard_begin, int64_t shard_end, Batch bt)
{
    __shared__ uint32_t wsum[RT / 32];
    bits += blockIdx.y * bt.bits_stride, flags = ws_of(flags, bt, blockIdx.y), hd = ws_of(hd, bt, blockIdx.y);
    blkcnt = ws_of(blkcnt, bt, blockIdx.y), blkoff = ws_of(blkoff, bt, blockIdx.y), slide += blockIdx.y;
    if (MODE == 1 && blkcnt[blockIdx.x] == 0) return;   // the counting pass found no qualifying run in this CTA's words
    const int64_t i = (int64_t)blockIdx.x * RT + threadIdx.x;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    uint32_t cnt = 0;
    int64_t rs[32 / 2], re[32 / 2];   // a word holds at most 16 run starts
    if (i < NW) {
        uint32_t w = bits[i];
        uint32_t prev = (i > 0) ? (bits[i - 1] >> 31) : (uint32_t)(hd->in.open != 0);
        uint32_t starts = w & ~((w << 1) | prev);
        if (Lmin > 32 && starts) {
            // a run that starts below another start of the same word ends inside the word: shorter than L_min.  Only the
            // topmost start can qualify (or reach the chunk end), and the start that sits on the shard's first sample is
            // emitted whatever its length.  (Dense masks -- probabilities that hover around the threshold -- otherwise cost
            // up to 16 walks per word.)
            uint32_t keep = 0x80000000u >> __clz(starts);
            const int64_t gb = shard_begin - t0 - i * 32;
            if (shard_begin >= 0 && gb >= 0 && gb < 32) keep |= 1u << gb;
            starts &= keep;
        }
        while (starts) {
            int s = __ffs(starts) - 1;
            starts &= starts - 1;
            int64_t g = i * 32 + s;
            int64_t e = find_end(bits, flags, NW, N, g);
            if (e < N || last_chunk) {
                if (e - g >= Lmin || t0 + g == shard_begin || t0 + e == shard_end) {
                    if (MODE == 1) rs[cnt] = g, re[cnt] = e;
                    cnt++;
                }
            } else if (MODE == 0) {   // touches the chunk end and the stream continues: becomes the carry
                hd->out_open = 1;
                hd->out_start = t0 + g;
            }
        }
    }
    // CTA-wide exclusive scan of cnt
    uint32_t incl = cnt;
    for (int o = 1; o < 32; o <<= 1) {
        uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) wsum[wid] = incl;
    __syncthreads();
    if (wid == 0) {
        uint32_t v = wsum[lane];
        uint32_t inc2 = v;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t u = __shfl_up_sync(0xffffffffu, inc2, o);
            if (lane >= o) inc2 += u;
        }
        wsum[lane] = inc2 - v;   // exclusive warp offsets
        if (MODE == 0 && lane == 31) blkcnt[blockIdx.x] = inc2;
    }
    __syncthreads();
    if (MODE == 1 && cnt) {
        int64_t slot = (int64_t)blkoff[blockIdx.x] + wsum[wid] + (incl - cnt);
        for (uint32_t q = 0; q < cnt; q++, slot++)
            if (slot < capacity) {
                gwi_trigger r;
                r.slide = slide, r.model_mask = 0, r.start = t0 + rs[q], r.end = t0 + re[q], r.peak_p = 0.f, r.mean_p = 0.f;
                out[slot] = r;
            }
    }
}

__global__ void k_scan(const uint32_t* __restrict__ blkcnt0, uint32_t* __restrict__ blkoff0, int64_t nblk, int64_t t0,
                       int slide0, Header* hd0, gwi_trigger* __restrict__ out, int capacity, int32_t* __restrict__ d_count,
                       int append0, Batch bt, int nslides)
{
    __shared__ uint32_t wsum[32];
    __shared__ uint32_t running;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  // the slides of a batch one after the other: the records of slide y + 1 go behind those of slide y (append)
  for (int y = 0; y < nslides; y++) {
    const uint32_t* blkcnt = ws_of(blkcnt0, bt, y);
    uint32_t* blkoff = ws_of(blkoff0, bt, y);
    Header* hd = ws_of(hd0, bt, y);
    const int slide = slide0 + y, append = y > 0 ? 1 : append0;
    if (threadIdx.x == 0) {
        hd->base = append ? *d_count : 0;
        running = (uint32_t)hd->base + (uint32_t)hd->head_emit;   // the carried run, if emitted, is the first new record
    }
    __syncthreads();
    for (int64_t base = 0; base < nblk; base += blockDim.x) {
        int64_t i = base + threadIdx.x;
        uint32_t v = (i < nblk) ? blkcnt[i] : 0, incl = v;
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += u;
        }
        if (lane == 31) wsum[wid] = incl;
        __syncthreads();
        if (wid == 0) {
            uint32_t x = wsum[lane], inc2 = x;
            for (int o = 1; o < 32; o <<= 1) {
                uint32_t u = __shfl_up_sync(0xffffffffu, inc2, o);
                if (lane >= o) inc2 += u;
            }
            wsum[lane] = inc2 - x;
        }
        __syncthreads();
        uint32_t excl = running + wsum[wid] + incl - v;
        if (i < nblk) blkoff[i] = excl;
        __syncthreads();
        if (threadIdx.x == blockDim.x - 1) running = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        hd->total = (int32_t)running;
        *d_count = (int32_t)running;
        if (hd->head_emit && hd->base < capacity && out) {
            gwi_trigger r;
            r.slide = slide, r.model_mask = 0, r.start = hd->in.start, r.end = t0 + hd->head_end, r.peak_p = 0.f, r.mean_p = 0.f;
            out[hd->base] = r;
        }
    }
    __syncthreads();
  }
}

// The scan of a batch of slides with the slides in parallel: per-slide totals (a warp per slide), their exclusive scan in
// slide order (one thread: the append order of the records is the slides' order), then the offsets inside every slide.
// Same results as k_scan walking the slides one after the other (57 us for 33 slides), in a tenth of the time.
__global__ void k_scan_batch(const uint32_t* __restrict__ blkcnt0, uint32_t* __restrict__ blkoff0, int64_t nblk, int64_t t0,
                             int slide0, Header* hd0, gwi_trigger* __restrict__ out, int capacity, int32_t* __restrict__ d_count,
                             int append0, Batch bt, int nslides)
{
    extern __shared__ uint32_t sbase[];                     // [nslides]: totals, then first record index of the slide
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5, nw = blockDim.x >> 5;
    for (int y = wid; y < nslides; y += nw) {
        const uint32_t* c = ws_of(blkcnt0, bt, y);
        uint32_t sum = 0;
        for (int64_t i = lane; i < nblk; i += 32) sum += c[i];
        for (int o = 16; o > 0; o >>= 1) sum += __shfl_xor_sync(0xffffffffu, sum, o);
        if (lane == 0) sbase[y] = sum + (uint32_t)ws_of(hd0, bt, y)->head_emit;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        uint32_t run = append0 ? (uint32_t)*d_count : 0u;
        for (int y = 0; y < nslides; y++) {
            const uint32_t t = sbase[y];
            sbase[y] = run;
            run += t;
        }
        *d_count = (int32_t)run;
    }
    __syncthreads();
    for (int y = wid; y < nslides; y += nw) {
        const uint32_t* c = ws_of(blkcnt0, bt, y);
        uint32_t* off = ws_of(blkoff0, bt, y);
        Header* hd = ws_of(hd0, bt, y);
        const uint32_t base = sbase[y];
        uint32_t running = base + (uint32_t)hd->head_emit;     // the carried run, if emitted, is the slide's first new record
        for (int64_t i0 = 0; i0 < nblk; i0 += 32) {
            const int64_t i = i0 + lane;
            const uint32_t v = i < nblk ? c[i] : 0u;
            uint32_t incl = v;
            for (int o = 1; o < 32; o <<= 1) {
                const uint32_t u = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += u;
            }
            if (i < nblk) off[i] = running + incl - v;
            running += __shfl_sync(0xffffffffu, incl, 31);
        }
        if (lane == 0) {
            hd->base = (int32_t)base;
            hd->total = (int32_t)running;
            if (hd->head_emit && (int)base < capacity && out) {
                gwi_trigger r;
                r.slide = slide0 + y, r.model_mask = 0, r.start = hd->in.start, r.end = t0 + hd->head_end, r.peak_p = 0.f, r.mean_p = 0.f;
                out[base] = r;
            }
        }
    }
}

// statistics of pbar over local [a,b): peak, sum (double), per-model mask.  The ST_THREADS threads of the CTA cooperate (a
// 1 s run is four samples per thread: the loads of a record are all in flight at once).
// mm (fused time-slide heads, gwi_heads.cu): one byte per sample with the models that exceeded the threshold on their own;
// P then holds the mean itself (M = 1)
__device__ void run_stats(const Ptrs& P, int M, float theta, int64_t a, int64_t b, float& peak, double& sum, int& mask,
                          const uint8_t* __restrict__ mm)
{
    __shared__ float s_peak[ST_THREADS];
    __shared__ double s_sum[ST_THREADS];
    __shared__ int s_mask[ST_THREADS];
    float pk = -1.f;
    double sm = 0.0;
    int mk = 0;
#pragma unroll 4
    for (int64_t i = a + threadIdx.x; i < b; i += blockDim.x) {
        float v = ens_mean(P, M, i);
        pk = fmaxf(pk, v);
        sm += (double)v;
        if (mm) mk |= mm[i];
        else
            for (int j = 0; j < M; j++) mk |= (P.p[j][i] > theta) << j;
    }
    s_peak[threadIdx.x] = pk, s_sum[threadIdx.x] = sm, s_mask[threadIdx.x] = mk;
    __syncthreads();
    for (int o = ST_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
            s_peak[threadIdx.x] = fmaxf(s_peak[threadIdx.x], s_peak[threadIdx.x + o]);
            s_sum[threadIdx.x] += s_sum[threadIdx.x + o];
            s_mask[threadIdx.x] |= s_mask[threadIdx.x + o];
        }
        __syncthreads();
    }
    peak = s_peak[0], sum = s_sum[0], mask = s_mask[0];
    __syncthreads();
}

__global__ void k_stats(Ptrs P, int M, float theta, int64_t N, int64_t t0, const Header* __restrict__ hd,
                        gwi_trigger* __restrict__ out, int capacity, Carry* carry, int64_t shard_begin, int64_t shard_end,
                        const uint8_t* __restrict__ mm, Batch bt)
{
    hd = ws_of(hd, bt, blockIdx.y);
    if (bt.row_stride) {                                   // (batches come from the fused heads: P holds the mean itself)
        P.p[0] += blockIdx.y * bt.row_stride;
        if (mm) mm += blockIdx.y * bt.row_stride;
    }
    if (carry) carry += blockIdx.y;
    const int nrec = min(hd->total, capacity);
    if ((int)blockIdx.x == (int)gridDim.x - 1) {   // last CTA: write the outgoing carry
        if (!carry) return;
        Carry c;
        c.open = hd->out_open, c.mask = 0, c.start = hd->out_start, c.sum = 0.0, c.peak = 0.f, c.pad = 0;
        if (c.open) {
            int64_t a = c.start > t0 ? c.start - t0 : 0;
            float pk; double sm; int mk;
            run_stats(P, M, theta, a, N, pk, sm, mk, mm);
            if (c.start < t0) pk = fmaxf(pk, hd->in.peak), sm += hd->in.sum, mk |= hd->in.mask;
            c.peak = pk, c.sum = sm, c.mask = mk;
        }
        if (threadIdx.x == 0) *carry = c;
        return;
    }
    if (!out) return;
    for (int r = hd->base + blockIdx.x; r < nrec; r += gridDim.x - 1) {
        int64_t s = out[r].start, e = out[r].end;
        int64_t a = s > t0 ? s - t0 : 0;
        float pk; double sm; int mk;
        run_stats(P, M, theta, a, e - t0, pk, sm, mk, mm);
        if (s < t0) pk = fmaxf(pk, hd->in.peak), sm += hd->in.sum, mk |= hd->in.mask;
        if (threadIdx.x == 0) {
            out[r].peak_p = pk;
            out[r].mean_p = (float)(sm / (double)(e - s));
            out[r].model_mask = mk | (s == shard_begin ? GWI_EDGE_LEFT : 0) | (e == shard_end ? GWI_EDGE_RIGHT : 0);
        }
    }
}

struct Layout {
    size_t hdr, bits, flags, cnt, off, total;
    int64_t NW, NB, NR;
};
Layout layout(int64_t N, bool with_bits = true)
{
    Layout L;
    L.NW = (N + 31) / 32;
    L.NB = (L.NW + WB - 1) / WB;
    L.NR = (L.NW + RT - 1) / RT;
    size_t o = 0;
    auto take = [&](size_t bytes) { size_t at = o; o += (bytes + 255) & ~(size_t)255; return at; };
    L.hdr = take(sizeof(Header));
    L.bits = with_bits ? take((size_t)(L.NW + 4) * 4) : 0;   // (a batch works on masks that the caller holds)
    L.flags = take((size_t)L.NB);
    L.cnt = take((size_t)L.NR * 4);
    L.off = take((size_t)L.NR * 4);
    L.total = o;
    return L;
}

} // namespace

extern "C" size_t gwi_carry_bytes(void) { return sizeof(Carry); }
extern "C" size_t gwi_triggers_workspace_bytes(int64_t N) { return N < 1 ? 0 : layout(N).total; }

extern "C" gwi_status gwi_ensemble_triggers(const float* const* d_prob, int32_t n_models, int64_t N, int64_t t0,
                                            float threshold, int64_t min_len, int32_t slide_id, int last_chunk,
                                            void* d_carry, gwi_trigger* d_triggers, int32_t capacity, int32_t* d_count,
                                            float* d_pbar, void* d_workspace, size_t workspace_bytes, void* cuda_stream)
{
    return gwi_post_run(d_prob, n_models, N, t0, threshold, min_len, slide_id, last_chunk, d_carry, d_triggers, capacity,
                        d_count, 0, d_pbar, d_workspace, workspace_bytes, (cudaStream_t)cuda_stream, -1, -1);
}

// ---- gwi_ensemble_triggers_static: the same call on a file-scope scratch array (no allocation anywhere in the call) ------
namespace {
constexpr size_t r256(size_t b) { return (b + 255) & ~(size_t)255; }
// layout(N).total, as a constant expression
constexpr size_t layout_total(int64_t N)
{
    return r256(sizeof(Header)) + r256((size_t)((N + 31) / 32 + 4) * 4) + r256((size_t)(((N + 31) / 32 + WB - 1) / WB)) +
           2 * r256((size_t)(((N + 31) / 32 + RT - 1) / RT) * 4);
}
constexpr size_t STATIC_SCRATCH_BYTES = layout_total(GWI_TRIGGERS_STATIC_MAX_N);
constexpr int STATIC_MAX_DEVICES = 64;
}
// In host code this name is a host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_triggers_scratch[STATIC_SCRATCH_BYTES];

extern "C" gwi_status gwi_ensemble_triggers_static(const float* const* d_prob, int32_t n_models, int64_t N, int64_t t0,
                                                   float threshold, int64_t min_len, int32_t slide_id, int last_chunk,
                                                   void* d_carry, gwi_trigger* d_triggers, int32_t capacity,
                                                   int32_t* d_count, float* d_pbar, void* cuda_stream)
{
    if (N > (int64_t)GWI_TRIGGERS_STATIC_MAX_N) {
        gwi_set_error("gwi_ensemble_triggers_static: N = %lld exceeds GWI_TRIGGERS_STATIC_MAX_N = %d (use gwi_ensemble_triggers "
                      "with a caller-owned workspace)", (long long)N, (int)GWI_TRIGGERS_STATIC_MAX_N);
        return GWI_ERR_CAPACITY;
    }
    if (N >= 1 && layout(N).total > STATIC_SCRATCH_BYTES) {   // cannot happen: layout_total restates layout()
        gwi_set_error("gwi_ensemble_triggers_static: internal scratch too small");
        return GWI_ERR_NOMEM;
    }
    // the array's device address, looked up once per device with that device current
    static void* scratch_of[STATIC_MAX_DEVICES] = {};
    int dev = -1;
    GWI_CUDA_CHECK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= STATIC_MAX_DEVICES) {
        gwi_set_error("gwi_ensemble_triggers_static: device %d out of range", dev);
        return GWI_ERR_UNSUPPORTED;
    }
    if (!scratch_of[dev]) {
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_triggers_scratch);
        if (e != cudaSuccess || !ptr) {
            gwi_set_error("gwi_ensemble_triggers_static: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return GWI_ERR_CUDA;
        }
        scratch_of[dev] = ptr;
    }
    void* ws = scratch_of[dev];
    // the array keeps the previous call's contents: the header starts from zero (the rest is fully rewritten before it is read)
    GWI_CUDA_CHECK(cudaMemsetAsync(ws, 0, r256(sizeof(Header)), (cudaStream_t)cuda_stream));
    return gwi_post_run(d_prob, n_models, N, t0, threshold, min_len, slide_id, last_chunk, d_carry, d_triggers, capacity,
                        d_count, 0, d_pbar, ws, STATIC_SCRATCH_BYTES, (cudaStream_t)cuda_stream, -1, -1);
}

// append != 0: *d_count holds the number of records already in d_triggers; the new ones go behind them.
static gwi_status post_from_bits(const Ptrs& P, int n_models, const uint8_t* d_mm, const uint32_t* bits, int64_t N, int64_t t0,
                                 float threshold, int64_t min_len, int32_t slide_id, int last_chunk, void* d_carry,
                                 gwi_trigger* d_triggers, int32_t capacity, int32_t* d_count, int append, char* ws, const Layout& L,
                                 cudaStream_t st, int64_t shard_begin, int64_t shard_end, int K = 1, Batch bt = Batch{0, 0, 0})
{
    // K > 1: the slides slide_id .. slide_id + K - 1 in the same six launches (bt: their strides)
    Header* hd = (Header*)(ws + L.hdr);
    uint8_t* flags = (uint8_t*)(ws + L.flags);
    uint32_t* cnt = (uint32_t*)(ws + L.cnt);
    uint32_t* off = (uint32_t*)(ws + L.off);
    k_blkflags<<<dim3((unsigned)L.NB, K), WB, 0, st>>>(bits, L.NW, flags, bt);
    k_head_run<<<K, 32, 0, st>>>(bits, flags, L.NW, N, t0, min_len, last_chunk, (const Carry*)d_carry, hd, shard_begin, shard_end, bt);
    k_runs<0><<<dim3((unsigned)L.NR, K), RT, 0, st>>>(bits, flags, L.NW, N, t0, min_len, last_chunk, slide_id, hd, cnt, off,
                                                      d_triggers, capacity, shard_begin, shard_end, bt);
    if (K > 1 && K <= 8192) k_scan_batch<<<1, 1024, (size_t)K * 4, st>>>(cnt, off, L.NR, t0, slide_id, hd, d_triggers, capacity, d_count, append, bt, K);
    else k_scan<<<1, 1024, 0, st>>>(cnt, off, L.NR, t0, slide_id, hd, d_triggers, capacity, d_count, append, bt, K);
    k_runs<1><<<dim3((unsigned)L.NR, K), RT, 0, st>>>(bits, flags, L.NW, N, t0, min_len, last_chunk, slide_id, hd, cnt, off,
                                                      d_triggers, capacity, shard_begin, shard_end, bt);
    // records are few: up to 128 CTAs per slide loop over them (32 per slide in a batch), the last one writes the carry
    int sgrid = K > 1 ? (capacity < 32 ? capacity + 1 : 33) : (capacity < 128 ? capacity + 1 : 129);
    k_stats<<<dim3(sgrid, K), ST_THREADS, 0, st>>>(P, n_models, threshold, N, t0, hd, d_triggers, capacity, (Carry*)d_carry, shard_begin,
                                                   shard_end, d_mm, bt);
    gwi_count_launch(6);
    GWI_CUDA_CHECK(cudaGetLastError());
    return GWI_OK;
}

// Clustering of one slide from a bit mask that the fused heads kernel (gwi_heads.cu) has written: d_bits = words of the
// mask (bit i of word w = sample 32 w + i, bits past N zero), d_pbar = the mean probability (run statistics), d_mm = the
// per-sample model bytes.  Same carry / append / shard semantics as gwi_post_run.
gwi_status gwi_post_run_bits(const uint32_t* d_bits, const float* d_pbar, const uint8_t* d_mm, int64_t N, int64_t t0, float threshold,
                             int64_t min_len, int32_t slide_id, int last_chunk, void* d_carry, gwi_trigger* d_triggers,
                             int32_t capacity, int32_t* d_count, int append, void* d_workspace, size_t workspace_bytes,
                             cudaStream_t st, int64_t shard_begin, int64_t shard_end)
{
    Layout L = layout(N);
    if (workspace_bytes < L.total || !d_bits || !d_pbar) {
        gwi_set_error("gwi_post_run_bits: bad argument / workspace");
        return GWI_ERR_ARG;
    }
    Ptrs P;
    P.p[0] = d_pbar;
    for (int j = 1; j < GWI_MAX_MODELS; j++) P.p[j] = nullptr;
    if (!d_carry) last_chunk = 1;
    return post_from_bits(P, 1, d_mm, d_bits, N, t0, threshold, min_len, slide_id, last_chunk, d_carry, d_triggers, capacity, d_count,
                          append, (char*)d_workspace, L, st, shard_begin, shard_end);
}

// The same for `nslides` slides at once: masks bits_stride words apart, means / model bytes row_stride apart, consecutive
// carry blocks; slide ids slide0 .. slide0 + nslides - 1; the records are appended slide after slide exactly as nslides
// calls of gwi_post_run_bits with append = 1 would leave them.
size_t gwi_post_batch_workspace_bytes(int64_t N, int nslides) { return N < 1 ? 0 : layout(N, false).total * (size_t)nslides; }

gwi_status gwi_post_run_bits_batch(const uint32_t* d_bits, int64_t bits_stride, const float* d_pbar, const uint8_t* d_mm, int64_t row_stride,
                                   int nslides, int64_t N, int64_t t0, float threshold, int64_t min_len, int32_t slide0, int last_chunk,
                                   void* d_carry, gwi_trigger* d_triggers, int32_t capacity, int32_t* d_count, int append,
                                   void* d_workspace, size_t workspace_bytes, cudaStream_t st, int64_t shard_begin, int64_t shard_end)
{
    Layout L = layout(N, false);
    if (workspace_bytes < L.total * (size_t)nslides || !d_bits || !d_pbar || !d_carry || nslides < 1 || nslides > 65535) {
        gwi_set_error("gwi_post_run_bits_batch: bad argument / workspace");
        return GWI_ERR_ARG;
    }
    Ptrs P;
    P.p[0] = d_pbar;
    for (int j = 1; j < GWI_MAX_MODELS; j++) P.p[j] = nullptr;
    return post_from_bits(P, 1, d_mm, d_bits, N, t0, threshold, min_len, slide0, last_chunk, d_carry, d_triggers, capacity, d_count,
                          append, (char*)d_workspace, L, st, shard_begin, shard_end, nslides, Batch{bits_stride, row_stride, L.total});
}

gwi_status gwi_post_run(const float* const* d_prob, int32_t n_models, int64_t N, int64_t t0, float threshold,
                        int64_t min_len, int32_t slide_id, int last_chunk, void* d_carry, gwi_trigger* d_triggers,
                        int32_t capacity, int32_t* d_count, int append, float* d_pbar, void* d_workspace,
                        size_t workspace_bytes, cudaStream_t st, int64_t shard_begin, int64_t shard_end)
{
    if (!d_prob || n_models < 1 || n_models > GWI_MAX_MODELS || N < 1 || capacity < 0 || !d_count || !d_workspace ||
        (capacity > 0 && !d_triggers) || ((uintptr_t)d_workspace & 255)) {
        gwi_set_error("gwi_ensemble_triggers: bad argument");
        return GWI_ERR_ARG;
    }
    Ptrs P;
    bool vec = ((uintptr_t)d_pbar & 15) == 0;
    for (int j = 0; j < n_models; j++) {
        if (!d_prob[j] || ((uintptr_t)d_prob[j] & 3)) {
            gwi_set_error("gwi_ensemble_triggers: d_prob[%d] null or misaligned", j);
            return GWI_ERR_ARG;
        }
        cudaPointerAttributes pa;
        if (cudaPointerGetAttributes(&pa, d_prob[j]) != cudaSuccess || pa.type != cudaMemoryTypeDevice) {
            cudaGetLastError();
            gwi_set_error("gwi_ensemble_triggers: d_prob[%d] is not a device pointer", j);
            return GWI_ERR_ARG;
        }
        P.p[j] = d_prob[j];
        vec = vec && (((uintptr_t)d_prob[j] & 15) == 0);
    }
    for (int j = n_models; j < GWI_MAX_MODELS; j++) P.p[j] = nullptr;
    Layout L = layout(N);
    if (workspace_bytes < L.total) {
        gwi_set_error("gwi_ensemble_triggers: workspace %zu < %zu bytes", workspace_bytes, L.total);
        return GWI_ERR_NOMEM;
    }
    if (!d_carry) last_chunk = 1;   // a chunk without carry is a whole stream
    char* ws = (char*)d_workspace;
    uint32_t* bits = (uint32_t*)(ws + L.bits);
    // one warp handles 128 samples per iteration; 148 SMs x 8 CTAs of 256 threads
    int64_t warps_needed = (L.NW * 32 + 127) / 128;
    int grid = (int)((warps_needed + 7) / 8);
    if (grid > 148 * 8) grid = 148 * 8;
    if (grid < 1) grid = 1;
    if (vec) k_mask<true><<<grid, 256, 0, st>>>(P, n_models, N, threshold, bits, L.NW, d_pbar);
    else k_mask<false><<<grid, 256, 0, st>>>(P, n_models, N, threshold, bits, L.NW, d_pbar);
    gwi_count_launch(1);
    return post_from_bits(P, n_models, nullptr, bits, N, t0, threshold, min_len, slide_id, last_chunk, d_carry, d_triggers, capacity,
                          d_count, append, ws, L, st, shard_begin, shard_end);
}
