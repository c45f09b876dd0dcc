// hmlfc_encode: the HMLFC encoder on the GPU (completed): RGB8 light field -> compressed stream.
//
//   PAPER.md:263  colour transform (YCoCg, lossless -> YCoCg-R)            } hmlfc_hierarchy (hmlfc_hierarchy.cu)
//   PAPER.md:200  RLFC hierarchy: RKV = filtered cluster, SRV = view - RKV  }
//   PAPER.md:227-248, Eqs. (1)-(2)  phase-shifted exhaustive block search     hmlfc_search (hmlfc_search.cu)
//   PAPER.md:249  replacement step: predictive SRV blocks -> residual blocks  } classify_kernel (this file)
//   PAPER.md:268  two block thresholds: "If the energy is less than the user  }
//                 set threshold the block is marked as insignificant and not stored"
//   PAPER.md:272  BISE of the stored blocks; PAPER.md:276 BFS linearisation, "we extend the application of BISE to
//                 encode the motion vector values"                             rank_kernel, compact_kernel, pack_kernel
//
// Readings: R5 (the even-even member of a 2 x 2 cluster is the reference), R8 (reference reads
// outside the image are 0), R10 (subtractive: e = P - R, additive: e = P + R), R11 (significant iff energy >= tau),
// R12 (open loop: residuals against the unthresholded reference), R13 (two flags per predictive block; policies
// adaptive / all / literal), R15 / R16 (BISE layouts, joint motion record).  The bytes written are "Stream format v1"
// of DESIGN.md section 4; nothing here is shared with the oracle's serialiser -- tests compare the two streams byte
// for byte.
#include "../../include/hmlfc.h"

#include <cuda_runtime.h>

#include <climits>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <chrono>
#include <cmath>
#include <vector>

namespace hmlfc {  // hmlfc_api.cu
cudaError_t scratch_pool(cudaMemPool_t *out);
cudaError_t scratch_pool_trim();
}

namespace {

constexpr int kThreads = 256;
constexpr uint32_t FULL = 0xffffffffu;
constexpr uint64_t kNoRec = ~0ull;

// one SRV plane-channel in stream order (levels top-down, planes row-major, channel innermost)
struct EncPc {
    uint64_t srv_off;    // element offset of the plane in d_srv
    uint64_t ref_off;    // element offset of the cluster's reference plane (predictive planes)
    uint64_t rec_off;    // element offset (int4 records) of the plane's search results; kNoRec for reference planes
    uint64_t flag_word;  // word offset of the plane-channel's `res` words in the flag section (`pred` words follow)
};

// second table, known after the value ranges are: BISE parameters and positions of the plane-channel's strings
struct EncPack {
    int32_t offset;      // value bias: stored value = offset + BISE value
    uint32_t pad;
    uint64_t val_base;   // first value of the plane-channel in the dense value array
    uint64_t mv_base;    // first record in the dense motion-record array
};

// one BISE string to pack: `count` values at src[base ..] -> bit string at word `out_word` of the section
struct PackJob {
    uint64_t base, count, out_word;
    uint32_t layout, m;
};

struct Stats {
    int vmin, vmax;
    unsigned n_res, n_pred;
};

template <int B>
__device__ __forceinline__ void load_row(const int16_t *__restrict__ p, int (&v)[B])
{
    if constexpr (B % 4 == 0) {
#pragma unroll
        for (int q = 0; q < B / 4; ++q) {
            const uint2 w = *reinterpret_cast<const uint2 *>(p + 4 * q);
            v[4 * q + 0] = (int)(int16_t)(w.x & 0xFFFFu); v[4 * q + 1] = (int)(int16_t)(w.x >> 16);
            v[4 * q + 2] = (int)(int16_t)(w.y & 0xFFFFu); v[4 * q + 3] = (int)(int16_t)(w.y >> 16);
        }
    } else if constexpr (B == 2) {
        const uint32_t w = *reinterpret_cast<const uint32_t *>(p);
        v[0] = (int)(int16_t)(w & 0xFFFFu); v[1] = (int)(int16_t)(w >> 16);
    } else {
#pragma unroll
        for (int i = 0; i < B; ++i) v[i] = p[i];
    }
}

// ---------------------------------------------------------------------------------------------------------------
// classify_kernel: one lane per block, one warp per 32-block flag word of one plane-channel.
//   energy E = sum |SRV block|; reference plane: res = E >= tau_ref;
//   predictive plane (R13), with Delta = the search's best SAD: adaptive: worth = E >= tau_res, pred = worth and Delta < E,
//   res = worth and (pred ? Delta : E) >= tau_res; all: pred = 1, res = Delta >= tau_res; literal: pred = res = Delta >= tau_res.
//   The stored values of a predicted block are its residual e = P -+ R(x+dx, y+dy) (replacement step; R10, R8,
//   R12); the SRV planes themselves stay untouched, so the thresholds can be changed and the kernel run again (tau bisection).
// Outputs: the `res` / `pred` flag words (ballots) straight into the stream's flag section, and per plane-channel the range of
// the stored values of its `res` blocks and the two block counts.
template <int B>
__global__ void __launch_bounds__(kThreads)
classify_kernel(const int16_t *__restrict__ srv, const int4 *__restrict__ rec, const EncPc *__restrict__ pcs, int Ws, int Ht, int nbx,
                int nblk, int fwords, int tau_ref, int tau_res, int policy, uint32_t *__restrict__ flags, Stats *__restrict__ stats)
{
    const int k = blockIdx.y;
    const int fw = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    if (fw >= fwords) return;
    const int lane = threadIdx.x & 31;
    const EncPc pc = pcs[k];
    const bool predictive = pc.rec_off != kNoRec;
    const int b = fw * 32 + lane;
    bool res = false, pred = false;
    int vmin = INT_MAX, vmax = INT_MIN;
    if (b < nblk) {
        const int by = b / nbx, bx = b - by * nbx;
        const int16_t *P = srv + pc.srv_off + (size_t)(by * B) * Ws + bx * B;
        int v[B][B];
        int E = 0;
#pragma unroll
        for (int j = 0; j < B; ++j) {
            load_row<B>(P + (size_t)j * Ws, v[j]);
#pragma unroll
            for (int i = 0; i < B; ++i) E += abs(v[j][i]);
        }
        if (!predictive) {
            res = E >= tau_ref;
        } else {
            const int4 r = rec[pc.rec_off + b];  // mode, dx, dy, Delta
            if (policy == 0) {
                const bool worth = E >= tau_res;
                pred = worth && r.w < E;
                res = worth && (pred ? r.w : E) >= tau_res;
            } else if (policy == 1) {
                pred = true;
                res = r.w >= tau_res;
            } else if (policy == 2) {
                res = r.w >= tau_res;
                pred = res;
            } else {  // 3: no motion compensation (the RLFC hierarchy alone): predictive planes coded intra
                res = E >= tau_res;
            }
            if (pred) {
                const int16_t *R = srv + pc.ref_off;
#pragma unroll
                for (int j = 0; j < B; ++j) {
                    const int y = by * B + j + r.z;
#pragma unroll
                    for (int i = 0; i < B; ++i) {
                        const int x = bx * B + i + r.y;
                        const int q = (x >= 0 && x < Ws && y >= 0 && y < Ht) ? (int)R[(size_t)y * Ws + x] : 0;
                        v[j][i] = r.x ? v[j][i] + q : v[j][i] - q;
                    }
                }
            }
        }
        if (res) {
#pragma unroll
            for (int j = 0; j < B; ++j)
#pragma unroll
                for (int i = 0; i < B; ++i) { vmin = min(vmin, v[j][i]); vmax = max(vmax, v[j][i]); }
        }
    }
    const uint32_t wres = __ballot_sync(FULL, res), wpred = __ballot_sync(FULL, pred);
    vmin = __reduce_min_sync(FULL, vmin);
    vmax = __reduce_max_sync(FULL, vmax);
    if (lane == 0) {
        flags[pc.flag_word + fw] = wres;
        if (predictive) flags[pc.flag_word + fwords + fw] = wpred;
        if (wres) {
            atomicMin(&stats[k].vmin, vmin);
            atomicMax(&stats[k].vmax, vmax);
            atomicAdd(&stats[k].n_res, (unsigned)__popc(wres));
        }
        if (wpred) atomicAdd(&stats[k].n_pred, (unsigned)__popc(wpred));
    }
}

// rank_kernel: one warp per flag map: exclusive prefix count of the set bits before every word (the payload / motion-record index
// of a block = rank of its word + popcount of the lower bits, "Using the block indices ...").
__global__ void __launch_bounds__(kThreads)
rank_kernel(const uint32_t *__restrict__ flags, const EncPc *__restrict__ pcs, int n_pc, int fwords, uint32_t *__restrict__ rank)
{
    const int job = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);  // (plane-channel, map)
    if (job >= 2 * n_pc) return;
    const int k = job >> 1, map = job & 1, lane = threadIdx.x & 31;
    const EncPc pc = pcs[k];
    if (map == 1 && pc.rec_off == kNoRec) return;
    const uint32_t *w = flags + pc.flag_word + (size_t)map * fwords;
    uint32_t *out = rank + ((size_t)k * 2 + map) * fwords;
    uint32_t run = 0;
    for (int base = 0; base < fwords; base += 32) {
        const int i = base + lane;
        const uint32_t c = i < fwords ? (uint32_t)__popc(w[i]) : 0u;
        uint32_t incl = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t n = __shfl_up_sync(FULL, incl, o);
            if (lane >= o) incl += n;
        }
        if (i < fwords) out[i] = run + incl - c;
        run += __shfl_sync(FULL, incl, 31);
    }
}

// compact_kernel: the stored values of every `res` block (minus the plane-channel's offset) and the joint motion record
// r = mode (2W+1)^2 + (dy+W)(2W+1) + (dx+W) of every `pred` block (R16), each to its rank position of the dense arrays.
template <int B>
__global__ void __launch_bounds__(kThreads)
compact_kernel(const int16_t *__restrict__ srv, const int4 *__restrict__ rec, const EncPc *__restrict__ pcs, const EncPack *__restrict__ pks,
               int Ws, int Ht, int nbx, int nblk, int fwords, int window, const uint32_t *__restrict__ flags, const uint32_t *__restrict__ rank,
               uint16_t *__restrict__ vals, uint32_t *__restrict__ mvs)
{
    const int k = blockIdx.y;
    const int fw = blockIdx.x * (kThreads / 32) + (threadIdx.x >> 5);
    if (fw >= fwords) return;
    const int lane = threadIdx.x & 31;
    const EncPc pc = pcs[k];
    const EncPack pk = pks[k];
    const bool predictive = pc.rec_off != kNoRec;
    const int b = fw * 32 + lane;
    const uint32_t below = (1u << lane) - 1u;
    const uint32_t wres = flags[pc.flag_word + fw];
    const uint32_t wpred = predictive ? flags[pc.flag_word + fwords + fw] : 0u;
    const bool pred = (wpred >> lane) & 1u;
    int4 m = make_int4(0, 0, 0, 0);
    if (pred) m = rec[pc.rec_off + b];  // mode, dx, dy, Delta
    if ((wres >> lane) & 1u) {
        const int by = b / nbx, bx = b - by * nbx;
        const int16_t *P = srv + pc.srv_off + (size_t)(by * B) * Ws + bx * B;
        const int16_t *R = srv + pc.ref_off;
        const uint64_t r = (uint64_t)rank[((size_t)k * 2) * fwords + fw] + (uint64_t)__popc(wres & below);
        uint16_t *o = vals + pk.val_base + r * (B * B);
#pragma unroll
        for (int j = 0; j < B; ++j) {
            int v[B];
            load_row<B>(P + (size_t)j * Ws, v);
            if (pred) {  // the residual of the replacement step, as in classify_kernel
                const int y = by * B + j + m.z;
#pragma unroll
                for (int i = 0; i < B; ++i) {
                    const int x = bx * B + i + m.y;
                    const int q = (x >= 0 && x < Ws && y >= 0 && y < Ht) ? (int)R[(size_t)y * Ws + x] : 0;
                    v[i] = m.x ? v[i] + q : v[i] - q;
                }
            }
#pragma unroll
            for (int i = 0; i < B; ++i) o[j * B + i] = (uint16_t)(v[i] - pk.offset);
        }
    }
    if (predictive) {
        if (pred) {
            const uint32_t nd = (uint32_t)(2 * window + 1);
            const uint64_t r = (uint64_t)rank[((size_t)k * 2 + 1) * fwords + fw] + (uint64_t)__popc(wpred & below);
            mvs[pk.mv_base + r] = (uint32_t)m.x * nd * nd + (uint32_t)(m.z + window) * nd + (uint32_t)(m.y + window);
        }
    }
    (void)nblk;
}

// reconstruct_sse_kernel: the encoder's own dense reconstruction at the current thresholds (what a decoder
// makes of the stream) and its squared error against the input:
//   acc_c = X_h + sum_L [ res ? stored : 0 ] + [ pred ? +-R'(x+dx, y+dy) : 0 ],  stored = P (reference / intra) or P -+ R(x+dx, y+dy),
//   R' = the reference sample AS STORED (0 where its block is insignificant or outside the image), R = the unthresholded one (R12);
//   then inverse YCoCg-R and clamp (R17, R19).  The sum of squared RGB differences feeds the PSNR of PAPER.md:366 / :375.
struct RecGeom {
    int h, U, V, Ws, Ht, nbx, fwords, shiftB;  // block = 1 << shiftB
    int UL[9];
    uint32_t kbase[9];                            // first plane-channel (stream order) of level L
    uint64_t top_off, x_ch;                       // element offset of the top-level RKV planes of channel 0 in d_x; channel stride
};

// One thread per block-row segment (B consecutive pixels of one block row of one view): the plane-channel descriptor, the flag words
// and the motion record of a (level, channel) are fetched once per B pixels.
template <int B>
__global__ void __launch_bounds__(kThreads)
reconstruct_sse_kernel(const uint8_t *__restrict__ lf, const int16_t *__restrict__ srv, const int16_t *__restrict__ xk, const int4 *__restrict__ rec,
                       const EncPc *__restrict__ pcs, const uint32_t *__restrict__ flags, RecGeom G, unsigned long long n_seg,
                       unsigned long long *__restrict__ sse)
{
    const unsigned long long g = (unsigned long long)blockIdx.x * kThreads + threadIdx.x;
    unsigned long long err = 0ull;
    if (g < n_seg) {
        const unsigned long long npx = (unsigned long long)G.Ws * G.Ht;
        const unsigned long long seg_per_view = npx / B;
        const int view = (int)(g / seg_per_view), seg = (int)(g - (unsigned long long)view * seg_per_view);
        const int v = view / G.U, u = view - v * G.U, t = seg / G.nbx, bx = seg - t * G.nbx, s0 = bx * B;
        const int b = (t >> G.shiftB) * G.nbx + bx;
        const int pix = t * G.Ws + s0;
        int a[3][B];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            load_row<B>(xk + G.top_off + (uint64_t)c * G.x_ch + (uint64_t)((v >> G.h) * G.UL[G.h] + (u >> G.h)) * npx + pix, a[c]);
            for (int L = 0; L < G.h; ++L) {
                const int pu = u >> L, pv = v >> L;
                const EncPc pc = pcs[G.kbase[L] + (uint32_t)(pv * G.UL[L] + pu) * 3u + c];
                const bool res = (flags[pc.flag_word + (b >> 5)] >> (b & 31)) & 1u;
                int P[B];
                load_row<B>(srv + pc.srv_off + pix, P);
                if (pc.rec_off != kNoRec && ((flags[pc.flag_word + G.fwords + (b >> 5)] >> (b & 31)) & 1u)) {
                    const int4 m = rec[pc.rec_off + b];
                    const uint64_t rflag = pcs[G.kbase[L] + (uint32_t)((pv & ~1) * G.UL[L] + (pu & ~1)) * 3u + c].flag_word;
                    const int y = t + m.z;
#pragma unroll
                    for (int i = 0; i < B; ++i) {
                        const int x = s0 + i + m.y;
                        int q = 0, qs = 0;
                        if (x >= 0 && x < G.Ws && y >= 0 && y < G.Ht) {
                            q = srv[pc.ref_off + (size_t)y * G.Ws + x];
                            const int rb = (y >> G.shiftB) * G.nbx + (x >> G.shiftB);
                            qs = ((flags[rflag + (rb >> 5)] >> (rb & 31)) & 1u) ? q : 0;
                        }
                        a[c][i] += (res ? (m.x ? P[i] + q : P[i] - q) : 0) + (m.x ? -qs : qs);
                    }
                } else if (res) {
#pragma unroll
                    for (int i = 0; i < B; ++i) a[c][i] += P[i];
                }
            }
        }
        const uint8_t *px = lf + ((unsigned long long)view * npx + pix) * 3ull;
#pragma unroll
        for (int i = 0; i < B; ++i) {
            const int tt = a[0][i] - (a[2][i] >> 1), Gc = a[2][i] + tt, Bc = tt - (a[1][i] >> 1), Rc = Bc + a[1][i];  // inverse YCoCg-R lifting
            const int dr = min(max(Rc, 0), 255) - (int)px[3 * i], dg = min(max(Gc, 0), 255) - (int)px[3 * i + 1],
                      db = min(max(Bc, 0), 255) - (int)px[3 * i + 2];
            err += (unsigned long long)(dr * dr + dg * dg + db * db);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) err += __shfl_xor_sync(FULL, err, o);
    if ((threadIdx.x & 31) == 0 && err) atomicAdd(sse, err);
}

// n <= 32 bits of v into an LSB-first 32-bit word string (zero-initialised; neighbouring groups share words)
__device__ __forceinline__ void or_bits(uint32_t *__restrict__ w, uint64_t pos, uint32_t v, uint32_t n)
{
    if (v == 0u || n == 0u) return;
    const uint64_t i = pos >> 5;
    const uint32_t sh = (uint32_t)(pos & 31u);
    atomicOr(&w[i], v << sh);
    if (sh + n > 32u) atomicOr(&w[i + 1], v >> (32u - sh));
}

// pack_kernel: BISE (layouts in DESIGN.md section 4), one lane per group.  plain: one m-bit value; trit: 8-bit
// T = sum t_k 3^k then five m-bit fields; quint: 7-bit Q = sum q_k 5^k then three m-bit fields; value = digit 2^m + low; the last
// group is padded with zero values.
template <typename T>
__global__ void __launch_bounds__(kThreads)
pack_kernel(const T *__restrict__ src, const PackJob *__restrict__ jobs, uint32_t *__restrict__ out)
{
    const PackJob jb = jobs[blockIdx.y];
    const uint32_t G = jb.layout == 0u ? 1u : (jb.layout == 1u ? 5u : 3u);
    const uint64_t ngroups = (jb.count + G - 1) / G;
    uint32_t *w = out + jb.out_word;
    const uint32_t m = jb.m, lmask = (1u << m) - 1u;
    for (uint64_t g = (uint64_t)blockIdx.x * kThreads + threadIdx.x; g < ngroups; g += (uint64_t)gridDim.x * kThreads) {
        if (jb.layout == 0u) {
            or_bits(w, g * m, (uint32_t)src[jb.base + g], m);
            continue;
        }
        const uint32_t hb = jb.layout == 1u ? 8u : 7u, radix = jb.layout == 1u ? 3u : 5u;
        const uint64_t pos = g * (uint64_t)(hb + G * m);
        uint32_t head = 0u, mul = 1u;
        for (uint32_t q = 0; q < G; ++q) {
            const uint64_t i = g * G + q;
            const uint32_t v = i < jb.count ? (uint32_t)src[jb.base + i] : 0u;
            head += (v >> m) * mul;
            mul *= radix;
            or_bits(w, pos + hb + (uint64_t)q * m, v & lmask, m);
        }
        or_bits(w, pos, head, hb);
    }
}

// ---------------------------------------------------------------------------------------------------------------- host side
void bise_choose(uint32_t N, uint32_t *layout, uint32_t *m)
{
    // cheapest bits per value, in 1/15 bit: plain 15 ceil(log2 N); trit (8 + 5m)/5 -> 24 + 15m; quint (7 + 3m)/3 -> 35 + 15m;
    // ties: plain, then trit, then quint (R15)
    if (N <= 1u) { *layout = 0u; *m = 0u; return; }
    uint32_t b = 0, mt = 0, mq = 0;
    while ((1ull << b) < (uint64_t)N) ++b;
    while ((3ull << mt) < (uint64_t)N) ++mt;
    while ((5ull << mq) < (uint64_t)N) ++mq;
    uint32_t best = 15u * b;
    *layout = 0u; *m = b;
    if (24u + 15u * mt < best) { best = 24u + 15u * mt; *layout = 1u; *m = mt; }
    if (35u + 15u * mq < best) { *layout = 2u; *m = mq; }
}

uint64_t bise_bits(uint32_t layout, uint32_t m, uint64_t count)
{
    if (layout == 0u) return count * m;
    if (layout == 1u) return ((count + 4) / 5) * (uint64_t)(8 + 5 * m);
    return ((count + 2) / 3) * (uint64_t)(7 + 3 * m);
}

void put16(uint8_t *p, uint32_t v) { p[0] = (uint8_t)v; p[1] = (uint8_t)(v >> 8); }
void put32(uint8_t *p, uint32_t v) { for (int i = 0; i < 4; ++i) p[i] = (uint8_t)(v >> (8 * i)); }
void put64(uint8_t *p, uint64_t v) { for (int i = 0; i < 8; ++i) p[i] = (uint8_t)(v >> (8 * i)); }
void putf(uint8_t *p, float f) { uint32_t u; memcpy(&u, &f, 4); put32(p, u); }
uint64_t up8(uint64_t x) { return (x + 7) & ~7ull; }

double now_ms() { return std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now().time_since_epoch()).count(); }

struct DevBuf {  // frees on scope exit
    void *p = nullptr;
    cudaStream_t st = nullptr;
    ~DevBuf() { if (p) cudaFreeAsync(p, st); }
    cudaError_t alloc(size_t bytes, cudaStream_t s)
    {
        st = s;
        cudaMemPool_t pool;
        cudaError_t e = hmlfc::scratch_pool(&pool);
        return e != cudaSuccess ? e : cudaMallocFromPoolAsync(&p, bytes ? bytes : 16, pool, s);
    }
    template <typename T> T *as() const { return static_cast<T *>(p); }
};

}  // namespace

#define ENC_CU(call)                                           \
    do {                                                       \
        cudaError_t e__ = (call);                              \
        if (e__ != cudaSuccess) { if (stats) stats->cuda_error = (int)e__; return e__ == cudaErrorMemoryAllocation ? HMLFC_E_NOMEM : HMLFC_E_CUDA; } \
    } while (0)

extern "C" void hmlfc_stream_free(uint8_t *h_stream) { free(h_stream); }

extern "C" int hmlfc_encode_release_scratch(void)
{
    return hmlfc::scratch_pool_trim() == cudaSuccess ? HMLFC_OK : HMLFC_E_CUDA;
}

// target_psnr < 0: encode at p's thresholds.  Otherwise ("encoding parameters are varied ... to achieve a similar
// compression quality"; W3, R24): bisection of tau_res in [0, 4096] with tau_ref = floor(tau_res / 2), at most max_iter
// steps, until the PSNR of the reconstruction is within tol of the target; the closest step wins.  Hierarchy and search run once
// (they do not depend on the thresholds, R12); every step is one classify pass + one reconstruction pass.
static int encode_impl(const uint8_t *d_lf, const hmlfc_encode_params_t *p_in, double target_psnr, double tol, int max_iter,
                       uint8_t **h_stream, size_t *len, hmlfc_encode_stats_t *stats, void *cuda_stream)
{
    if (stats) memset(stats, 0, sizeof(*stats));
    const double t_begin = now_ms();
    if (!d_lf || !p_in || !h_stream || !len) return HMLFC_E_INVALID;
    hmlfc_encode_params_t prm = *p_in;
    hmlfc_encode_params_t *p = &prm;
    const int U = p->U, V = p->V, Ws = p->Ws, Ht = p->Ht, h = p->height, B = p->block, W = p->window;
    if (U < 1 || V < 1 || Ws < 1 || Ht < 1 || h < 1 || p->tau_ref < 0 || p->tau_res < 0 || p->policy < 0 || p->policy > 3) return HMLFC_E_INVALID;
    if (h > 8 || (B != 2 && B != 4 && B != 8) || W < 0 || W > 64 || Ws % B || Ht % B || Ws % 4 || (long long)U * V > (1 << 24))
        return HMLFC_E_UNSUPPORTED;  // what hmlfc_load accepts and hmlfc_hierarchy needs
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const size_t npx = (size_t)Ws * Ht;
    const int nbx = Ws / B, nby = Ht / B, nblk = nbx * nby, fwords = (nblk + 31) / 32;
    int UL[10], VL[10];
    size_t lvl_plane0[10];  // first SRV plane of level L inside a channel of d_srv
    int64_t ns = 0, nx = 0;
    for (int L = 0; L <= h; ++L) {
        UL[L] = (U + (1 << L) - 1) >> L; VL[L] = (V + (1 << L) - 1) >> L;
        if (L < h) { lvl_plane0[L] = (size_t)ns; ns += (int64_t)UL[L] * VL[L]; }
        if (L >= 1) nx += (int64_t)UL[L] * VL[L];
    }
    const uint64_t n_pc = (uint64_t)ns * 3;
    if (n_pc > 65535u * 16u) return HMLFC_E_UNSUPPORTED;
    const int n_top = UL[h] * VL[h];

    cudaEvent_t ev[6];
    for (auto &e : ev) ENC_CU(cudaEventCreate(&e));
    struct EvGuard { cudaEvent_t *e; ~EvGuard() { for (int i = 0; i < 6; ++i) cudaEventDestroy(e[i]); } } evg{ev};

    // ---- 1. colour + hierarchy
    DevBuf srv, xk;
    ENC_CU(srv.alloc((size_t)3 * ns * npx * sizeof(int16_t), st));
    ENC_CU(xk.alloc((size_t)3 * nx * npx * sizeof(int16_t), st));
    ENC_CU(cudaEventRecord(ev[0], st));
    int rc = hmlfc_hierarchy(d_lf, U, V, Ws, Ht, h, srv.as<int16_t>(), xk.as<int16_t>(), st);
    if (rc != HMLFC_OK) return rc;
    ENC_CU(cudaEventRecord(ev[1], st));

    // ---- 2. roles (R5) and the phase-shifted search of every predictive plane
    // pairs of level L in plane order; the records of (channel c, level L, pair j) start at ((pair0[L] * 3 + c * npairs[L]) + j) * nblk
    std::vector<std::vector<int32_t>> pairs(h);
    std::vector<std::vector<int32_t>> pair_of(h);  // plane -> pair index or -1
    std::vector<uint64_t> rec0(h);                 // first record (in blocks) of level L, channel 0
    uint64_t n_rec = 0;
    for (int L = 0; L < h; ++L) {
        pair_of[L].assign((size_t)UL[L] * VL[L], -1);
        for (int pv = 0; pv < VL[L]; ++pv)
            for (int pu = 0; pu < UL[L]; ++pu)
                if ((pu | pv) & 1) {
                    pair_of[L][(size_t)pv * UL[L] + pu] = (int32_t)(pairs[L].size() / 2);
                    pairs[L].push_back(pv * UL[L] + pu);
                    pairs[L].push_back((pv & ~1) * UL[L] + (pu & ~1));
                }
        rec0[L] = n_rec;
        n_rec += (uint64_t)3 * (pairs[L].size() / 2) * nblk;
    }
    DevBuf rec, dpairs;
    ENC_CU(rec.alloc((size_t)n_rec * sizeof(int4), st));
    size_t pair_words = 0;
    for (int L = 0; L < h; ++L) pair_words += pairs[L].size();
    ENC_CU(dpairs.alloc(pair_words * sizeof(int32_t), st));
    {
        size_t o = 0;
        for (int L = 0; L < h; ++L) {
            if (!pairs[L].empty())
                ENC_CU(cudaMemcpyAsync(dpairs.as<int32_t>() + o, pairs[L].data(), pairs[L].size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
            const int np = (int)(pairs[L].size() / 2);
            for (int c = 0; c < 3; ++c)
                for (int j0 = 0; j0 < np; j0 += 65535) {
                    const int nj = np - j0 < 65535 ? np - j0 : 65535;
                    rc = hmlfc_search(srv.as<int16_t>() + ((size_t)c * ns + lvl_plane0[L]) * npx, dpairs.as<int32_t>() + o + 2 * (size_t)j0, nj, Ws, Ht,
                                      B, W, reinterpret_cast<int32_t *>(rec.as<int4>() + rec0[L] + ((uint64_t)c * np + j0) * nblk), st);
                    if (rc != HMLFC_OK) return rc;
                }
            o += pairs[L].size();
        }
    }
    ENC_CU(cudaEventRecord(ev[2], st));

    // ---- 3. plane-channel table in stream order (BFS from the top of the tree), flag section layout
    std::vector<EncPc> pcs((size_t)n_pc);
    std::vector<uint8_t> is_pred((size_t)n_pc);
    uint64_t flag_words = 0;
    {
        size_t k = 0;
        for (int L = h - 1; L >= 0; --L)
            for (int pv = 0; pv < VL[L]; ++pv)
                for (int pu = 0; pu < UL[L]; ++pu)
                    for (int c = 0; c < 3; ++c, ++k) {
                        const size_t pl = (size_t)pv * UL[L] + pu;
                        const int pj = pair_of[L][pl];
                        EncPc e;
                        e.srv_off = ((size_t)c * ns + lvl_plane0[L] + pl) * npx;
                        e.ref_off = ((size_t)c * ns + lvl_plane0[L] + (size_t)(pv & ~1) * UL[L] + (pu & ~1)) * npx;
                        e.rec_off = pj < 0 ? kNoRec : rec0[L] + ((uint64_t)c * (pairs[L].size() / 2) + (uint64_t)pj) * nblk;
                        e.flag_word = flag_words;
                        flag_words += (uint64_t)fwords * (pj < 0 ? 1 : 2);
                        is_pred[k] = pj >= 0;
                        pcs[k] = e;
                    }
    }
    DevBuf dpcs, dflags, dstats, drank;
    ENC_CU(dpcs.alloc(pcs.size() * sizeof(EncPc), st));
    ENC_CU(dflags.alloc((size_t)flag_words * 4, st));
    ENC_CU(dstats.alloc((size_t)n_pc * sizeof(Stats), st));
    ENC_CU(drank.alloc((size_t)n_pc * 2 * fwords * sizeof(uint32_t), st));
    ENC_CU(cudaMemcpyAsync(dpcs.p, pcs.data(), pcs.size() * sizeof(EncPc), cudaMemcpyHostToDevice, st));
    std::vector<Stats> hstats((size_t)n_pc);
    const std::vector<Stats> stats0((size_t)n_pc, Stats{INT_MAX, INT_MIN, 0u, 0u});
    DevBuf dsse;
    ENC_CU(dsse.alloc(sizeof(unsigned long long), st));

    // ---- 4. thresholds + replacement; plane-channels in chunks of 65535 (grid.y)
    const unsigned gx = (unsigned)((fwords + kThreads / 32 - 1) / (kThreads / 32));
    auto threshold = [&](int tau_ref, int tau_res) -> cudaError_t {
        cudaError_t e = cudaMemcpyAsync(dstats.p, stats0.data(), stats0.size() * sizeof(Stats), cudaMemcpyHostToDevice, st);
        if (e != cudaSuccess) return e;
        for (uint64_t k0 = 0; k0 < n_pc; k0 += 65535) {
            const unsigned nk = (unsigned)(n_pc - k0 < 65535 ? n_pc - k0 : 65535);
            const dim3 grid(gx, nk);
#define CLASSIFY(BB) classify_kernel<BB><<<grid, kThreads, 0, st>>>(srv.as<int16_t>(), rec.as<int4>(), dpcs.as<EncPc>() + k0, Ws, Ht, nbx, nblk, fwords, \
                                                                    tau_ref, tau_res, p->policy, dflags.as<uint32_t>(), dstats.as<Stats>() + k0)
            if (B == 2) CLASSIFY(2); else if (B == 4) CLASSIFY(4); else CLASSIFY(8);
#undef CLASSIFY
        }
        return cudaGetLastError();
    };
    // squared error of the reconstruction at the thresholds last applied (synchronises)
    RecGeom geo{};
    geo.h = h; geo.U = U; geo.V = V; geo.Ws = Ws; geo.Ht = Ht; geo.nbx = nbx; geo.fwords = fwords; geo.shiftB = B == 2 ? 1 : (B == 4 ? 2 : 3);
    {
        uint32_t kb = 0;
        for (int L = h - 1; L >= 0; --L) { geo.kbase[L] = kb; kb += (uint32_t)(UL[L] * VL[L]) * 3u; }
        for (int L = 0; L <= h; ++L) geo.UL[L] = UL[L];
        geo.top_off = (uint64_t)(nx - n_top) * npx; geo.x_ch = (uint64_t)nx * npx;
    }
    const unsigned long long n_lf_px = (unsigned long long)U * V * npx;
    auto measure_sse = [&](unsigned long long *out) -> cudaError_t {
        cudaError_t e = cudaMemsetAsync(dsse.p, 0, sizeof(unsigned long long), st);
        if (e != cudaSuccess) return e;
        const unsigned long long n_seg = n_lf_px / (unsigned long long)B;
        const unsigned gs = (unsigned)((n_seg + kThreads - 1) / kThreads);
#define RECON(BB) reconstruct_sse_kernel<BB><<<gs, kThreads, 0, st>>>(d_lf, srv.as<int16_t>(), xk.as<int16_t>(), rec.as<int4>(), dpcs.as<EncPc>(), \
                                                                     dflags.as<uint32_t>(), geo, n_seg, dsse.as<unsigned long long>())
        if (B == 2) RECON(2); else if (B == 4) RECON(4); else RECON(8);
#undef RECON
        if ((e = cudaGetLastError()) != cudaSuccess) return e;
        if ((e = cudaMemcpyAsync(out, dsse.p, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st)) != cudaSuccess) return e;
        return cudaStreamSynchronize(st);
    };
    auto psnr_of = [&](unsigned long long se) -> double {  // 10 log10(255^2 / MSE) over all RGB bytes
        if (se == 0ull) return INFINITY;
        return 10.0 * log10(255.0 * 255.0 / ((double)se / (double)(n_lf_px * 3ull)));
    };
    int n_steps = 0;
    unsigned long long sse = 0ull;
    if (target_psnr >= 0.0) {
        int lo = 0, hi = 4096, best_tau = -1;
        double best_q = 0.0;
        for (int it = 0; it < max_iter; ++it) {
            const int mid = (lo + hi) / 2;
            ENC_CU(threshold(mid / 2, mid));
            ENC_CU(measure_sse(&sse));
            ++n_steps;
            const double q = psnr_of(sse);
            if (best_tau < 0 || fabs(q - target_psnr) < fabs(best_q - target_psnr)) { best_tau = mid; best_q = q; }
            if (fabs(q - target_psnr) <= tol || hi - lo <= 1) break;
            if (q > target_psnr) lo = mid; else hi = mid;
        }
        prm.tau_res = best_tau;
        prm.tau_ref = best_tau / 2;
    }
    ENC_CU(threshold(p->tau_ref, p->tau_res));
    rank_kernel<<<(unsigned)((2 * n_pc + kThreads / 32 - 1) / (kThreads / 32)), kThreads, 0, st>>>(dflags.as<uint32_t>(), dpcs.as<EncPc>(), (int)n_pc, fwords,
                                                                                                  drank.as<uint32_t>());
    ENC_CU(cudaGetLastError());
    ENC_CU(cudaEventRecord(ev[3], st));
    ENC_CU(cudaMemcpyAsync(hstats.data(), dstats.p, hstats.size() * sizeof(Stats), cudaMemcpyDeviceToHost, st));
    ENC_CU(cudaStreamSynchronize(st));
    ENC_CU(measure_sse(&sse));  // quality of the stream about to be written

    // ---- 5. directory: value range -> BISE layout, string positions
    uint32_t mv_layout, mv_m;
    const uint32_t mvN = 2u * (uint32_t)(2 * W + 1) * (uint32_t)(2 * W + 1);
    bise_choose(mvN, &mv_layout, &mv_m);
    std::vector<EncPack> pks((size_t)n_pc);
    std::vector<PackJob> vjobs, mjobs;
    struct Dirent { int32_t offset; uint32_t N, layout, m; uint64_t pay_bitoff, mv_bitoff; };
    std::vector<Dirent> dir((size_t)n_pc);
    uint64_t pay_bits = 0, mv_bits = 0, n_vals = 0, n_mvs = 0, max_vgroups = 1, max_mgroups = 1, tot_res = 0;
    for (size_t k = 0; k < n_pc; ++k) {
        Stats &s = hstats[k];
        if (s.n_res == 0) { s.vmin = 0; s.vmax = 0; }
        Dirent &d = dir[k];
        d.offset = s.vmin;
        d.N = (uint32_t)(s.vmax - s.vmin + 1);
        bise_choose(d.N, &d.layout, &d.m);
        const uint64_t cnt = (uint64_t)s.n_res * B * B;
        d.pay_bitoff = pay_bits;
        pay_bits = (pay_bits + bise_bits(d.layout, d.m, cnt) + 31) & ~31ull;
        d.mv_bitoff = mv_bits;
        mv_bits = (mv_bits + bise_bits(mv_layout, mv_m, s.n_pred) + 31) & ~31ull;
        pks[k] = EncPack{d.offset, 0u, n_vals, n_mvs};
        if (cnt && d.m + (d.layout ? 1u : 0u) > 0u) {
            vjobs.push_back(PackJob{n_vals, cnt, d.pay_bitoff / 32, d.layout, d.m});
            const uint64_t G = d.layout == 0 ? 1 : (d.layout == 1 ? 5 : 3);
            if ((cnt + G - 1) / G > max_vgroups) max_vgroups = (cnt + G - 1) / G;
        }
        if (s.n_pred) {
            mjobs.push_back(PackJob{n_mvs, s.n_pred, d.mv_bitoff / 32, mv_layout, mv_m});
            const uint64_t G = mv_layout == 0 ? 1 : (mv_layout == 1 ? 5 : 3);
            if ((s.n_pred + G - 1) / G > max_mgroups) max_mgroups = (s.n_pred + G - 1) / G;
        }
        n_vals += cnt;
        n_mvs += s.n_pred;
        tot_res += s.n_res;
    }
    const uint64_t rkv_bytes = (uint64_t)n_top * npx * 5;
    const uint64_t off_rkv = 160, off_dir = up8(off_rkv + rkv_bytes), off_flags = up8(off_dir + n_pc * 48);
    const uint64_t off_payload = up8(off_flags + flag_words * 4), off_mv = up8(off_payload + pay_bits / 8 + 8);
    const uint64_t total = up8(off_mv + mv_bits / 8 + 8);

    // ---- 6. dense values / records in rank order, then the BISE strings
    DevBuf dpks, dvals, dmvs, dpay, dmvbits, dvjobs, dmjobs;
    ENC_CU(dpks.alloc(pks.size() * sizeof(EncPack), st));
    ENC_CU(dvals.alloc((size_t)n_vals * sizeof(uint16_t), st));
    ENC_CU(dmvs.alloc((size_t)n_mvs * sizeof(uint32_t), st));
    ENC_CU(dpay.alloc((size_t)(pay_bits / 8 + 8), st));
    ENC_CU(dmvbits.alloc((size_t)(mv_bits / 8 + 8), st));
    ENC_CU(dvjobs.alloc(vjobs.size() * sizeof(PackJob), st));
    ENC_CU(dmjobs.alloc(mjobs.size() * sizeof(PackJob), st));
    ENC_CU(cudaMemcpyAsync(dpks.p, pks.data(), pks.size() * sizeof(EncPack), cudaMemcpyHostToDevice, st));
    if (!vjobs.empty()) ENC_CU(cudaMemcpyAsync(dvjobs.p, vjobs.data(), vjobs.size() * sizeof(PackJob), cudaMemcpyHostToDevice, st));
    if (!mjobs.empty()) ENC_CU(cudaMemcpyAsync(dmjobs.p, mjobs.data(), mjobs.size() * sizeof(PackJob), cudaMemcpyHostToDevice, st));
    ENC_CU(cudaMemsetAsync(dpay.p, 0, (size_t)(pay_bits / 8 + 8), st));
    ENC_CU(cudaMemsetAsync(dmvbits.p, 0, (size_t)(mv_bits / 8 + 8), st));
    ENC_CU(cudaEventRecord(ev[4], st));
    for (uint64_t k0 = 0; k0 < n_pc; k0 += 65535) {
        const unsigned nk = (unsigned)(n_pc - k0 < 65535 ? n_pc - k0 : 65535);
        const dim3 grid(gx, nk);
#define COMPACT(BB) compact_kernel<BB><<<grid, kThreads, 0, st>>>(srv.as<int16_t>(), rec.as<int4>(), dpcs.as<EncPc>() + k0, dpks.as<EncPack>() + k0, Ws, Ht, nbx, nblk, \
                                                                  fwords, W, dflags.as<uint32_t>(), drank.as<uint32_t>() + k0 * 2 * fwords, dvals.as<uint16_t>(), dmvs.as<uint32_t>())
        if (B == 2) COMPACT(2); else if (B == 4) COMPACT(4); else COMPACT(8);
#undef COMPACT
    }
    // grid = (CTAs per string, strings): the strings differ in length, so a string gets at most 32 CTAs that stride over its groups
    // (a CTA whose first group is beyond the string leaves at once)
    auto pack_grid_x = [](uint64_t groups) { uint64_t g = (groups + kThreads - 1) / kThreads; return (unsigned)(g > 32 ? 32 : g); };
    for (size_t j0 = 0; j0 < vjobs.size(); j0 += 65535) {
        const unsigned nj = (unsigned)(vjobs.size() - j0 < 65535 ? vjobs.size() - j0 : 65535);
        pack_kernel<uint16_t><<<dim3(pack_grid_x(max_vgroups), nj), kThreads, 0, st>>>(dvals.as<uint16_t>(), dvjobs.as<PackJob>() + j0, dpay.as<uint32_t>());
    }
    for (size_t j0 = 0; j0 < mjobs.size(); j0 += 65535) {
        const unsigned nj = (unsigned)(mjobs.size() - j0 < 65535 ? mjobs.size() - j0 : 65535);
        pack_kernel<uint32_t><<<dim3(pack_grid_x(max_mgroups), nj), kThreads, 0, st>>>(dmvs.as<uint32_t>(), dmjobs.as<PackJob>() + j0, dmvbits.as<uint32_t>());
    }
    ENC_CU(cudaGetLastError());
    ENC_CU(cudaEventRecord(ev[5], st));

    const double t_assemble = now_ms();
    // ---- 7. stream assembly on the host (header, raw top-level RKVs, directory) + the three device-built sections
    uint8_t *s = static_cast<uint8_t *>(calloc((size_t)total, 1));
    if (!s) return HMLFC_E_NOMEM;
    struct HostGuard { uint8_t *p; ~HostGuard() { free(p); } } hg{s};
    memcpy(s, "HMLF", 4);
    put16(s + 4, 1); put16(s + 6, 160);
    put32(s + 8, (uint32_t)U); put32(s + 12, (uint32_t)V); put32(s + 16, (uint32_t)Ws); put32(s + 20, (uint32_t)Ht);
    put32(s + 24, (uint32_t)h); put32(s + 28, (uint32_t)B); put32(s + 32, (uint32_t)W); put32(s + 36, 3);
    put32(s + 40, (uint32_t)p->tau_ref); put32(s + 44, (uint32_t)p->tau_res);
    s[48] = 1; s[49] = 0; s[50] = 0; s[51] = (uint8_t)p->policy;
    s[52] = p->background[0]; s[53] = p->background[1]; s[54] = p->background[2];
    putf(s + 56, p->uv_origin[0]); putf(s + 60, p->uv_origin[1]); putf(s + 64, p->uv_step[0]); putf(s + 68, p->uv_step[1]);
    putf(s + 72, p->st_origin[0]); putf(s + 76, p->st_origin[1]); putf(s + 80, p->st_step[0]); putf(s + 84, p->st_step[1]);
    putf(s + 88, p->z_st);
    put64(s + 96, p->seed); put64(s + 104, n_pc);
    put64(s + 112, off_rkv); put64(s + 120, off_dir); put64(s + 128, off_flags); put64(s + 136, off_payload); put64(s + 144, off_mv);
    put64(s + 152, total);
    {
        // top-level RKVs = the last U_h V_h planes of every channel of d_x: Y as uint8, Co / Cg as int16 (R6, R20)
        std::vector<int16_t> top((size_t)n_top * npx);
        uint8_t *o = s + off_rkv;
        for (int c = 0; c < 3; ++c) {
            ENC_CU(cudaMemcpyAsync(top.data(), xk.as<int16_t>() + ((size_t)c * nx + (size_t)(nx - n_top)) * npx, top.size() * sizeof(int16_t),
                                   cudaMemcpyDeviceToHost, st));
            ENC_CU(cudaStreamSynchronize(st));
            if (c == 0) for (size_t i = 0; i < top.size(); ++i) *o++ = (uint8_t)top[i];
            else for (size_t i = 0; i < top.size(); ++i) { put16(o, (uint32_t)(uint16_t)top[i]); o += 2; }
        }
    }
    for (size_t k = 0; k < n_pc; ++k) {
        uint8_t *e = s + off_dir + k * 48;
        put32(e, (uint32_t)dir[k].offset); put32(e + 4, dir[k].N); put32(e + 8, hstats[k].n_res); put32(e + 12, hstats[k].n_pred);
        put64(e + 16, pcs[k].flag_word * 4); put64(e + 24, dir[k].pay_bitoff); put64(e + 32, dir[k].mv_bitoff);
        e[40] = (uint8_t)dir[k].layout; e[41] = (uint8_t)dir[k].m; e[42] = is_pred[k];
    }
    ENC_CU(cudaMemcpyAsync(s + off_flags, dflags.p, (size_t)flag_words * 4, cudaMemcpyDeviceToHost, st));
    ENC_CU(cudaMemcpyAsync(s + off_payload, dpay.p, (size_t)(pay_bits / 8), cudaMemcpyDeviceToHost, st));
    ENC_CU(cudaMemcpyAsync(s + off_mv, dmvbits.p, (size_t)(mv_bits / 8), cudaMemcpyDeviceToHost, st));
    ENC_CU(cudaStreamSynchronize(st));
    if (stats) {
        float ms = 0.f;
        cudaEventElapsedTime(&ms, ev[0], ev[1]); stats->ms_hierarchy = ms;
        cudaEventElapsedTime(&ms, ev[1], ev[2]); stats->ms_search = ms;
        cudaEventElapsedTime(&ms, ev[2], ev[3]); stats->ms_classify = ms;
        cudaEventElapsedTime(&ms, ev[4], ev[5]); stats->ms_pack = ms;
        stats->ms_wall = (float)(now_ms() - t_begin);
        stats->ms_assemble = (float)(now_ms() - t_assemble);
        stats->sse = (int64_t)sse;
        stats->psnr = psnr_of(sse);
        stats->tau_ref = p->tau_ref;
        stats->tau_res = p->tau_res;
        stats->bisection_steps = n_steps;
        stats->n_plane_channels = (int64_t)n_pc;
        stats->n_res_blocks = (int64_t)tot_res;
        stats->n_pred_blocks = (int64_t)n_mvs;
        stats->n_search_blocks = (int64_t)n_rec;
        stats->kernel_launches = 0;  // filled below
        int nl = h;  // hierarchy
        for (int L = 0; L < h; ++L) nl += 3 * (int)((pairs[L].size() / 2 + 65534) / 65535);
        nl += 2 * (int)((n_pc + 65534) / 65535) + 1 + (int)((vjobs.size() + 65534) / 65535) + (int)((mjobs.size() + 65534) / 65535);
        stats->kernel_launches = nl;
    }
    hg.p = nullptr;
    *h_stream = s;
    *len = (size_t)total;
    return HMLFC_OK;
}

extern "C" int hmlfc_encode(const uint8_t *d_lf, const hmlfc_encode_params_t *p, uint8_t **h_stream, size_t *len,
                            hmlfc_encode_stats_t *stats, void *cuda_stream)
{
    return encode_impl(d_lf, p, -1.0, 0.0, 0, h_stream, len, stats, cuda_stream);
}

extern "C" int hmlfc_encode_psnr(const uint8_t *d_lf, const hmlfc_encode_params_t *p, double target_psnr, double tol, int max_iter,
                                 uint8_t **h_stream, size_t *len, hmlfc_encode_stats_t *stats, void *cuda_stream)
{
    if (!(target_psnr >= 0.0) || !(tol >= 0.0) || max_iter < 1 || !std::isfinite(target_psnr)) {
        if (stats) memset(stats, 0, sizeof(*stats));
        return HMLFC_E_INVALID;
    }
    return encode_impl(d_lf, p, target_psnr, tol, max_iter, h_stream, len, stats, cuda_stream);
}
