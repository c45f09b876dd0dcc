// hmlfc_decode, warp-cooperative form (sm_100a): the tree walk of 32 random coordinates regrouped into
// uniform batches of work.
//
// What is computed is exactly DESIGN.md section 3: per coordinate and channel
//   acc = topRKV + sum_L [ stored_p(s,t)  (+|-)  stored_r(s+dx, t+dy) ].
// For uniformly random coordinates every test of that walk (block significant? block predicted? reference
// block significant?) is taken by a different subset of the lanes, so a thread-per-coordinate kernel runs
// with ~8 of 32 lanes active (profiles/r01c_final.md).  Here each lane still classifies ITS coordinate with uniform control
// flow, but everything behind a set flag becomes a task on small per-warp stacks in shared memory; tasks are executed 32 at a time by
// all lanes (a stack is drained whenever it holds >= 32 tasks, so only the last batch of a warp is partial).  Values are
// accumulated with shared-memory atomics into the destination's (Y, Co, Cg) cell; the owning lane finishes with the inverse
// colour transform and the staged 96-byte store.  Integer arithmetic only: bit-exact by construction against the per-thread
// kernel and the oracle.
//
// Two kernels:
//   decode_brec_kernel   on the BLOCK RECORDS hmlfc_load builds (hmlfc_device.cuh): one 32-byte slot per level says what the plane
//                        holds for the sample and where; value / motion / lookup tasks cover the three channels.  The default.
//   decode_queue_kernel  on the stream's own BISE strings: kMode 0 (eager: flag records and descriptors of the three channels up front,
//                        tasks carry them) and 1 (lazy: one flag sector per level, tasks fetch descriptor and rank); its kSubpel / kCs
//                        instantiations read half-pel (R28) and chroma-subsampled (R18) streams, which have no block records; kDense
//                        1 / 2 generate whole views / blocks for block sizes other than 4.
#include "hmlfc_kernels.cuh"

#include <type_traits>

namespace hmlfc {

namespace {

constexpr int kThreads = 256, kWarps = kThreads / 32;
constexpr int kCap = 64;  // per stack: < 32 left over + <= 32 pushed per round
// runs of 32 coordinates per warp of the block-record kernel.  Two runs sharing the stacks (the last, partial batches paid once per 64
// coordinates) measured SLOWER: cfg2 11.8 against 16.9 G px/s -- 5 KB more shared memory per CTA is L1 taken away, and the second run's
// slot loads wait behind the first run's pushes.
constexpr int kBrecSets = 1;

struct DigitLut {
    uint16_t v[384];
};

// digits of the packed trit / quint words: T -> t0 | t1<<2 | .. | t4<<8, Q -> q0 | q1<<3 | q2<<6
constexpr DigitLut make_digit_lut()
{
    DigitLut l{};
    for (int T = 0; T < 256; ++T) {
        int x = T, p = 0;
        for (int k = 0; k < 5; ++k) { p |= (x % 3) << (2 * k); x /= 3; }
        l.v[T] = (uint16_t)p;
    }
    for (int Q = 0; Q < 128; ++Q) {
        int x = Q, p = 0;
        for (int k = 0; k < 3; ++k) { p |= (x % 5) << (3 * k); x /= 5; }
        l.v[256 + Q] = (uint16_t)p;
    }
    return l;
}

__device__ const DigitLut g_dq_digit_lut = make_digit_lut();

// (shared memory is L1 taken away: this kernel's loads live on L1 hits of descriptors, slots and neighbouring fields, so the stacks stay small)
template <int kLookups, int kSets>
struct WarpQT {
    uint4 vq[kCap];              // value tasks
    uint4 mq[kCap];              // motion tasks
    uint4 rq[kLookups];          // reference lookups (block records only)
    int acc[kSets * 32 * 4];     // {Y, Co, Cg, -} per coordinate of the warp
    uint32_t xy[kSets * 32];     // s | t << 16 of the warp's coordinates
};
using WarpQ = WarpQT<1, 1>;

// BISE decode_at (bit layout in DESIGN.md section 4) of value i of the string that starts at word `base`
// of `words`, without control flow: plain = groups of one value with an empty digit word, so lanes holding tasks of
// different layouts do not serialise.  A group (<= 58 bits from any bit offset) lies in three consecutive words; they
// are fetched as TWO aligned 64-bit loads (every lane-load of a random coordinate costs a sector-gather whatever its
// width, profiles/r01_gather_probe.md), then the digit word and the value's m-bit field are cut out with funnel shifts.
__device__ __forceinline__ uint32_t bise_at(const uint32_t *__restrict__ words, uint32_t base, uint32_t i, uint32_t layout, uint32_t m,
                                            const uint16_t *__restrict__ lut)
{
    const bool plain = layout == 0u, trit = layout == 1u;
    const uint32_t G = plain ? 1u : (trit ? 5u : 3u), hb = plain ? 0u : (trit ? 8u : 7u);
    const uint32_t g = plain ? i : (trit ? (__umulhi(i, 0xCCCCCCCDu) >> 2) : (__umulhi(i, 0xAAAAAAABu) >> 1));
    const uint32_t k = i - G * g;
    const uint32_t gb = g * (hb + G * m);
    const uint32_t wi = base + (gb >> 5), sh = gb & 31u;   // absolute word index of the group's first bit
    const uint2 *p2 = reinterpret_cast<const uint2 *>(words + (wi & ~1u));
    const uint2 A = __ldg(p2), B = __ldg(p2 + 1);          // words [wi & ~1, +4): covers wi .. wi + 2 (16 bytes of slack follow the string)
    const bool odd = (wi & 1u) != 0u;
    const uint32_t w0 = odd ? A.y : A.x, w1 = odd ? B.x : A.y, w2 = odd ? B.y : B.x;
    const uint32_t head = __funnelshift_r(w0, w1, sh) & ((1u << hb) - 1u);  // plain: 0 bits -> 0, the quint table maps 0 to digit 0
    const uint32_t pos = sh + hb + k * m;                  // payload groups (<= 63 bits): the field ends inside w2
    uint32_t lo = pos < 32u ? w0 : (pos < 64u ? w1 : w2), hi = pos < 32u ? w1 : (pos < 64u ? w2 : 0u);
    if (pos + m > 96u) {  // motion records of wide windows (W = 51..54: trit m = 13, 73-bit groups): the field's own two words
        const uint32_t *f = words + base + ((gb + hb + k * m) >> 5);
        lo = __ldg(f);
        hi = __ldg(f + 1);
    }
    const uint32_t low = __funnelshift_r(lo, hi, pos & 31u) & ((1u << m) - 1u);
    const uint32_t dig = ((uint32_t)lut[(trit ? 0u : 256u) + head] >> (k * (trit ? 2u : 3u))) & (trit ? 3u : 7u);
    return (dig << m) | low;
}

constexpr uint32_t kSignBit = 1u << 23;  // value task: subtract (additive / "phase-shifted" mode, R10)

// push one task per flagged lane on a warp stack; cnt is warp-uniform
__device__ __forceinline__ void push(uint4 *stack, int &cnt, bool flag, uint4 task, uint32_t lane_lt)
{
    const uint32_t m = __ballot_sync(0xffffffffu, flag);
    if (flag) stack[cnt + __popc(m & lane_lt)] = task;
    cnt += __popc(m);
}

// index of the 32-bit word with the res bits of plane-channel k's group g: Y / Co in the slot's fourth record, Cg in its own
__device__ __forceinline__ size_t resbits_word(const DevStream &S, uint32_t k, uint32_t g)
{
    const uint32_t p = __umulhi(k, 0xAAAAAAABu) >> 1, c = k - 3u * p;  // k / 3, k % 3
    return (((size_t)p * (size_t)S.fgroups + (size_t)g) * 4u + (c == 2u ? 2u : 3u)) * 4u + (c == 1u ? 1u : 0u);
}

// execute the top n (<= 32) value tasks: rank of the block (S4) and BISE decode_at of its value (S5)
template <typename Q>
__device__ __forceinline__ void drain_values(const DevStream &S, Q &q, int &vcnt, int n, int lane, const uint16_t *lut)
{
    __syncwarp();
    if (lane < n) {
        const uint4 t = q.vq[vcnt - n + lane];
        const uint4 d = ldg(S.pc + t.x);
        const uint32_t rank0 = __ldg(reinterpret_cast<const uint32_t *>(S.flagrec + flag_index(S, t.x, t.y)) + 1);  // res blocks before the group
        const uint32_t idx = ((rank0 + ((t.z >> 8) & 63u)) << (2 * S.logB)) + (t.z & 63u);
        int val = pc_offset(d.w) + (int)bise_at(S.pay, d.y, idx, pc_layout(d.w), pc_m(d.w), lut);
        if (t.z & kSignBit) val = -val;
        atomicAdd(&q.acc[t.z >> 24], val);
    }
    vcnt -= n;
    __syncwarp();
}

// execute the top n (<= 32) motion tasks: decode the record (S6), locate the reference sample (S7) and, where
// the reference block is significant, push its value task
template <typename Q>
__device__ __forceinline__ void drain_motion(const DevStream &S, Q &q, int &mcnt, int &vcnt, int n, int lane,
                                             uint32_t lane_lt, const uint16_t *lut)
{
    __syncwarp();
    bool has = false;
    uint4 vt = make_uint4(0u, 0u, 0u, 0u);
    if (lane < n) {
        const uint4 t = q.mq[mcnt - n + lane];
        const uint4 d = ldg(S.pc + t.x);
        const uint32_t prank0 = __ldg(reinterpret_cast<const uint32_t *>(S.flagrec + flag_index(S, t.x, t.y)) + 3);  // pred blocks before the group
        const uint32_t rec = bise_at(S.mv, d.z, prank0 + ((t.w >> 8) & 31u), S.mv_layout, S.mv_m, lut);
        int mode, dx, dy;
        mv_unpack(S, rec, mode, dx, dy);
        const uint32_t dest = t.w & 0xFFu;
        const uint32_t xy = q.xy[dest >> 2];
        const int rx = (int)(xy & 0xFFFFu) + dx, ry = (int)(xy >> 16) + dy;
        if ((unsigned)rx < (unsigned)S.Ws && (unsigned)ry < (unsigned)S.Ht) {  // R8: outside the image reads 0
            const int b = (ry >> S.logB) * S.nbx + (rx >> S.logB);
            const uint32_t g = (uint32_t)(b >> 5), bit = 1u << (b & 31);
            const uint32_t bits = __ldg(reinterpret_cast<const uint32_t *>(S.flagrec) + resbits_word(S, t.z, g));
            has = (bits & bit) != 0u;
            const uint32_t kin = (uint32_t)(((ry & (S.B - 1)) << S.logB) + (rx & (S.B - 1)));
            vt = make_uint4(t.z, g, kin | ((uint32_t)__popc(bits & (bit - 1u)) << 8) | (mode ? kSignBit : 0u) | (dest << 24), 0u);
        }
    }
    mcnt -= n;
    __syncwarp();
    push(q.vq, vcnt, has, vt, lane_lt);
}

// The same two steps for tasks that carry everything the classification already fetched (eager form, below):
//   motion task  {MV word base, record index, reference plane-channel, destination}
//   value task   {payload word base, value index, offset|layout|m|sign|destination}
// execute the top n (<= 32) value tasks: S5 of the path
template <typename Q>
__device__ __forceinline__ void drain_values_eager(const DevStream &S, Q &q, int &vcnt, int n, int lane, const uint16_t *lut)
{
    __syncwarp();
    if (lane < n) {
        const uint4 t = q.vq[vcnt - n + lane];
        int val = pc_offset(t.z) + (int)bise_at(S.pay, t.x, t.y, pc_layout(t.z), pc_m(t.z), lut);
        if (t.z & kSignBit) val = -val;
        atomicAdd(&q.acc[t.z >> 24], val);
    }
    vcnt -= n;
    __syncwarp();
}

// execute the top n (<= 32) motion tasks: decode the record (S6), locate the reference sample (S7) and, where
// the reference block is significant, push its value task
template <bool kSubpel, bool kCs, typename Q>
__device__ __forceinline__ void drain_motion_eager(const DevStream &S, Q &q, int &mcnt, int &vcnt, int n, int lane,
                                             uint32_t lane_lt, const uint16_t *lut)
{
    __syncwarp();
    bool has = false;
    uint4 vt = make_uint4(0u, 0u, 0u, 0u);
    if (lane < n) {
        const uint4 t = q.mq[mcnt - n + lane];
        const uint32_t rec = bise_at(S.mv, t.x, t.y, S.mv_layout, S.mv_m, lut);
        int mode, dx, dy;
        mv_unpack(S, rec, mode, dx, dy);
        const uint32_t xy = q.xy[t.w >> 2];
        // the channel's own geometry: (kCs, R18) Co / Cg live at half resolution, sample (s >> 1, t >> 1)
        const int csh = (kCs && (t.w & 3u) != 0u) ? 1 : 0;
        const int px = (int)(xy & 0xFFFFu) >> csh, py = (int)(xy >> 16) >> csh, cW = S.Ws >> csh, cH = S.Ht >> csh, cnbx = csh ? S.nbx_c : S.nbx;
        if (kSubpel) {
            // half-pel offsets (R28): the reference value is the mean of the 1 / 2 / 4 stored samples around the position, rounded
            // half up -- the sum has to be complete before it is rounded, so the lane looks the samples up itself (no value tasks)
            const int x2 = 2 * px + dx, y2 = 2 * py + dy;
            const int x0 = x2 >> 1, y0 = y2 >> 1, fx = x2 & 1, fy = y2 & 1;
            const uint4 rd = ldg(S.pc + t.z);
            int sum = 0;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                if (((j & 1) && !fx) || ((j >> 1) && !fy)) continue;
                const int rx = x0 + (j & 1), ry = y0 + (j >> 1);
                if ((unsigned)rx >= (unsigned)cW || (unsigned)ry >= (unsigned)cH) continue;  // R8
                const int b = (ry >> S.logB) * cnbx + (rx >> S.logB);
                const uint4 fr = ldg(S.flagrec + flag_index(S, t.z, (uint32_t)(b >> 5)));
                const uint32_t bit = 1u << (b & 31);
                if (!(fr.x & bit)) continue;
                const uint32_t rank = fr.y + (uint32_t)__popc(fr.x & (bit - 1u));
                const uint32_t kin = (uint32_t)(((ry & (S.B - 1)) << S.logB) + (rx & (S.B - 1)));
                sum += pc_offset(rd.w) + (int)bise_at(S.pay, rd.y, (rank << (2 * S.logB)) + kin, pc_layout(rd.w), pc_m(rd.w), lut);
            }
            const int k = fx + fy, qv = (sum + k) >> k;  // rounding term n / 2 = 0, 1, 2 = k
            atomicAdd(&q.acc[t.w], mode ? -qv : qv);
        } else {
            const int rx = px + dx, ry = py + dy;
            if ((unsigned)rx < (unsigned)cW && (unsigned)ry < (unsigned)cH) {  // R8: outside the image reads 0
                const int b = (ry >> S.logB) * cnbx + (rx >> S.logB);
                const uint4 rd = ldg(S.pc + t.z);
                const uint4 fr = ldg(S.flagrec + flag_index(S, t.z, (uint32_t)(b >> 5)));
                const uint32_t bit = 1u << (b & 31);
                has = (fr.x & bit) != 0u;
                const uint32_t rank = fr.y + (uint32_t)__popc(fr.x & (bit - 1u));
                const uint32_t kin = (uint32_t)(((ry & (S.B - 1)) << S.logB) + (rx & (S.B - 1)));
                vt = make_uint4(rd.y, (rank << (2 * S.logB)) + kin, (rd.w & 0x3FFFFFu) | (mode ? kSignBit : 0u) | (t.w << 24), 0u);
            }
        }
    }
    mcnt -= n;
    __syncwarp();
    if (!kSubpel) push(q.vq, vcnt, has, vt, lane_lt);
}

// The same steps on the block records (hmlfc_device.cuh; kMode 2).  One task covers the three channels:
//   value task   {word of the sample's first field, what (below), offset Y | offset Co << 16, offset Cg}
//                what = bit | present << 5 | wanted << 8 | subtract << 11 | wY << 14 | wCo << 18 | wCg << 22 | destination lane << 26
//                (present: the channels whose fields follow each other from that bit on; wanted: those to accumulate)
//   motion task  {word of the block's first motion record, bit | pred mask << 5 | destination lane << 8, reference plane}
//   lookup task  {reference plane, rx | ry << 16, channels | subtract << 3 | destination lane << 8}: channels whose motion records point at
//                the same reference sample share the lookup and, where the reference block holds them, the value task
__device__ __forceinline__ uint32_t value_what(uint32_t bit, uint32_t present, uint32_t wanted, uint32_t sub, uint4 pb, uint32_t lane)
{
    return bit | (present << 5) | (wanted << 8) | (sub << 11) | ((pb.y & 0xFu) << 14) | (((pb.y >> 8) & 0xFu) << 18) | (((pb.y >> 16) & 0xFu) << 22) | (lane << 26);
}

template <bool kCg, typename Q>
__device__ __forceinline__ void drain_values_brec(const DevStream &S, Q &q, int &vcnt, int n, int lane)
{
    __syncwarp();
    if (lane < n) {
        const uint4 t = q.vq[vcnt - n + lane];
        const uint32_t sh = t.y & 31u, present = (t.y >> 5) & 7u, wanted = (t.y >> 8) & 7u, sub = (t.y >> 11) & 7u;
        const uint32_t w[3] = {(t.y >> 14) & 15u, (t.y >> 18) & 15u, (t.y >> 22) & 15u};
        const int off[3] = {(int)(int16_t)(t.z & 0xFFFFu), (int)(int16_t)(t.z >> 16), (int)(int16_t)(t.w & 0xFFFFu)};
        const uint32_t span = ((present & 1u) ? w[0] : 0u) + ((present & 2u) ? w[1] : 0u) + ((present & 4u) ? w[2] : 0u);
        const BrecWindow win = brec_window<kCg>(S.brec, ((unsigned long long)t.x << 5) | sh, span);
        int *acc = q.acc + (t.y >> 26) * 4;
        uint32_t pos = sh;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if (!((present >> c) & 1u)) continue;
            if ((wanted >> c) & 1u) {
                const int val = off[c] + (int)brec_window_field(win, pos, w[c]);
                atomicAdd(acc + c, ((sub >> c) & 1u) ? -val : val);
            }
            pos += w[c];
        }
    }
    vcnt -= n;
    __syncwarp();
}

// reference lookups: slot and descriptor of the reference plane -> value task for the channels its block holds
template <bool kCg, typename Q>
__device__ __forceinline__ void drain_lookups_brec(const DevStream &S, Q &q, int &rcnt, int &vcnt, int n, int lane, uint32_t lane_lt)
{
    __syncwarp();
    bool has = false;
    uint4 vt = make_uint4(0u, 0u, 0u, 0u);
    if (lane < n) {
        const uint4 t = q.rq[rcnt - n + lane];
        const int rx = (int)(t.y & 0xFFFFu), ry = (int)(t.y >> 16);
        const int b = (ry >> S.logB) * S.nbx + (rx >> S.logB);
        uint4 sa, sb;
        if (kCg) ldcg256(S.bslot + ((size_t)t.x * (size_t)S.fgroups + (size_t)(b >> 5)) * 2u, sa, sb);
        else ldg256(S.bslot + ((size_t)t.x * (size_t)S.fgroups + (size_t)(b >> 5)) * 2u, sa, sb);
        const uint4 pb = ldg(S.pb + t.x);
        const BrecPos r = brec_locate(S, sa, sb, 1u << (b & 31), pb);
        const uint32_t wanted = (t.z & 7u) & r.res;
        has = wanted != 0u;
        const uint32_t kin = (uint32_t)(((ry & (S.B - 1)) << S.logB) + (rx & (S.B - 1)));
        const unsigned long long pos = r.bit + brec_sample_offset(r, pb, kin);
        vt = make_uint4((uint32_t)(pos >> 5), value_what((uint32_t)pos & 31u, r.res, wanted, (t.z >> 3) & 7u, pb, (t.z >> 8) & 63u), pb.z, pb.w);
    }
    rcnt -= n;
    __syncwarp();
    push(q.vq, vcnt, has, vt, lane_lt);
}

// motion records of a block (S6), reference sample of every predicted channel (S7) -> lookup tasks
template <bool kCg, typename Q>
__device__ __forceinline__ void drain_motion_brec(const DevStream &S, Q &q, int &mcnt, int &rcnt, int &vcnt, int n, int lane, uint32_t lane_lt)
{
    __syncwarp();
    uint32_t rem = 0u, sub = 0u;
    int px[3] = {0, 0, 0}, py[3] = {0, 0, 0};
    uint4 t = make_uint4(0u, 0u, 0u, 0u);
    if (lane < n) {
        t = q.mq[mcnt - n + lane];
        const uint32_t sh = t.y & 31u, pred = (t.y >> 5) & 7u;
        const BrecWindow win = brec_window<kCg>(S.brec, ((unsigned long long)t.x << 5) | sh, popc(pred) * S.mv_w);
        const uint32_t xy = q.xy[(t.y >> 8) & 63u];
        uint32_t pos = sh;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            if (!((pred >> c) & 1u)) continue;
            int mode, dx, dy;
            mv_unpack(S, brec_window_field(win, pos, S.mv_w), mode, dx, dy);
            pos += S.mv_w;
            px[c] = (int)(xy & 0xFFFFu) + dx; py[c] = (int)(xy >> 16) + dy;
            if (mode) sub |= 1u << c;
            if ((unsigned)px[c] < (unsigned)S.Ws && (unsigned)py[c] < (unsigned)S.Ht) rem |= 1u << c;  // R8: outside the image reads 0
        }
    }
    mcnt -= n;
    __syncwarp();
    // one lookup per distinct reference sample: the first channel and every channel whose motion record points at the same sample (usually
    // all: the channels of a block move together), then the same for what is left (a pass through the motion stack for the few stragglers
    // would run whole 32-lane batches for a handful of tasks)
#pragma unroll
    for (int round = 0; round < 3; ++round) {
        if (!__any_sync(0xffffffffu, rem != 0u)) break;
        const int c0 = (rem & 1u) ? 0 : (rem & 2u) ? 1 : 2;
        const int x0 = c0 == 0 ? px[0] : c0 == 1 ? px[1] : px[2], y0 = c0 == 0 ? py[0] : c0 == 1 ? py[1] : py[2];
        uint32_t grp = 0u;
#pragma unroll
        for (int c = 0; c < 3; ++c)
            if (((rem >> c) & 1u) && px[c] == x0 && py[c] == y0) grp |= 1u << c;
        push(q.rq, rcnt, rem != 0u, make_uint4(t.z, (uint32_t)x0 | ((uint32_t)y0 << 16), grp | (sub << 3) | (((t.y >> 8) & 63u) << 8), 0u), lane_lt);
        rem &= ~grp;
        if (rcnt >= 32) {
            drain_lookups_brec<kCg>(S, q, rcnt, vcnt, 32, lane, lane_lt);
            if (vcnt >= 32) drain_values_brec<kCg>(S, q, vcnt, 32, lane);
        }
    }
}

template <int kMode, typename Q>
__device__ __forceinline__ void drain_v(const DevStream &S, Q &q, int &vcnt, int n, int lane, const uint16_t *lut)
{
    if (kMode == 1) drain_values(S, q, vcnt, n, lane, lut);
    else drain_values_eager(S, q, vcnt, n, lane, lut);
}

template <int kMode, bool kSubpel, bool kCs, typename Q>
__device__ __forceinline__ void drain_m(const DevStream &S, Q &q, int &mcnt, int &vcnt, int n, int lane, uint32_t lane_lt, const uint16_t *lut)
{
    if (kMode == 1) drain_motion(S, q, mcnt, vcnt, n, lane, lane_lt, lut);
    else drain_motion_eager<kSubpel, kCs>(S, q, mcnt, vcnt, n, lane, lane_lt, lut);
}

// kDense: the coordinates are not read but generated -- sample i is pixel i mod (Ws Ht) (row-major) of view views[i / (Ws Ht)]
// (hmlfc_decode_views: whole views, no 16-byte coordinate per sample, neighbouring lanes in neighbouring pixels).
// kLazy: the classification reads one flag sector per level and the tasks fetch descriptor and rank themselves (fewest sectors per sample: for
// streams the L2 holds, where the sector rate binds); otherwise it reads the three channels' flag records and descriptors up front and the
// tasks carry them (one dependent load less per task: for streams in HBM, where every access is a DRAM access either way and latency binds).
// kSubpel (eager form only): streams with half-pel motion offsets, see drain_motion_eager.
// kCs (eager form only): chroma-subsampled streams -- the Co / Cg channels of a sample are classified on their own block grid.
template <int kDense, int kMode, bool kSubpel = false, bool kCs = false>  // kDense 0: coordinates read; 1: whole views; 2: whole B x B blocks (u, v, bx, by) = blocks[i / B^2], written [n][B][B][3]
__global__ void __launch_bounds__(kThreads, 5)
decode_queue_kernel(const DevStream S, const int4 *__restrict__ coords, long long n, uint8_t *__restrict__ out,
                    unsigned long long *oob, int out_aligned)
{
    __shared__ WarpQ wq[kWarps];
    __shared__ uint16_t lut[384];
    for (int k = threadIdx.x; k < 384; k += kThreads) lut[k] = g_dq_digit_lut.v[k];
    __syncthreads();

    const int lane = threadIdx.x & 31;
    const uint32_t lane_lt = (1u << lane) - 1u;
    auto &q = wq[threadIdx.x >> 5];
    const long long i = (long long)blockIdx.x * kThreads + threadIdx.x;
    const bool present = i < n;
    int4 c4 = make_int4(0, 0, 0, 0);
    if (kDense == 2) {
        if (present) {
            const int bb = S.B * S.B;
            const long long blk = i / bb;
            const int k = (int)(i - blk * bb);
            const int4 q = __ldg(coords + blk);
            const int ky = k >> S.logB;
            c4 = make_int4(q.x, q.y, q.z * S.B + (k - (ky << S.logB)), q.w * S.B + ky);
            if ((unsigned)q.z >= (unsigned)S.nbx || (unsigned)q.w >= (unsigned)S.nby) c4.z = -1;
        }
    } else if (kDense == 1) {
        if (present) {
            const long long npx = (long long)S.Ws * S.Ht;
            const long long view = i / npx;
            const int pix = (int)(i - view * npx);
            const int2 uv = __ldg(reinterpret_cast<const int2 *>(coords) + view);
            const int y = pix / S.Ws;
            c4 = make_int4(uv.x, uv.y, pix - y * S.Ws, y);
        }
    } else {
#ifdef HMLFC_DECODE_CS
        if (present) c4 = __ldcs(coords + i);
#else
        if (present) c4 = __ldg(coords + i);
#endif
    }
    const bool valid = present && (unsigned)c4.x < (unsigned)S.U && (unsigned)c4.y < (unsigned)S.V &&
                       (unsigned)c4.z < (unsigned)S.Ws && (unsigned)c4.w < (unsigned)S.Ht;
    if (present && !valid) atomicAdd(oob, 1ull);
    const int u = c4.x, v = c4.y, x = c4.z, y = c4.w;
    const int h = S.h;

    // S3 root term: one 64-bit load; the cell starts at the top-level RKV sample
    short4 root = make_short4(0, 0, 0, 0);
    if (valid) root = ldg(S.rkv + ((size_t)((v >> h) * S.UH + (u >> h)) * (size_t)S.Ht + (size_t)y) * (size_t)S.Ws + (size_t)x);
    q.acc[lane * 4 + 0] = root.x;
    q.acc[lane * 4 + 1] = root.y;
    q.acc[lane * 4 + 2] = root.z;
    q.xy[lane] = (uint32_t)x | ((uint32_t)y << 16);

    const int b = valid ? (y >> S.logB) * S.nbx + (x >> S.logB) : 0;
    const uint32_t bit = 1u << (b & 31);
    const uint32_t fg = (uint32_t)(b >> 5);
    const uint32_t kin = (uint32_t)(((y & (S.B - 1)) << S.logB) + (x & (S.B - 1)));
    // (kCs) the same for the sample's chroma position (x >> 1, y >> 1) on the chroma block grid
    const int xc = x >> 1, yc = y >> 1;
    const int b_c = (kCs && valid) ? (yc >> S.logB) * S.nbx_c + (xc >> S.logB) : 0;
    const uint32_t bit_c = kCs ? 1u << (b_c & 31) : bit, fg_c = kCs ? (uint32_t)(b_c >> 5) : fg;
    const uint32_t kin_c = kCs ? (uint32_t)(((yc & (S.B - 1)) << S.logB) + (xc & (S.B - 1))) : kin;
    const uint32_t bit0 = bit, kin0 = kin;
    int vcnt = 0, mcnt = 0;

    constexpr bool kLazy = kMode == 1;
    if (kLazy) {
        // S4, first look, for (up to) four levels at a time: the six flag words of the block's group in each level's plane, one 32-byte
        // sector per level (the second half of the plane's 64-byte slot: the Cg record {res, rank, pred, rank} and {res Y, res Co, pred Y,
        // pred Co}).  The addresses depend on the coordinate alone, so the levels' loads are in flight together: one memory round trip
        // where a level-by-level walk takes h.  What a level contributes is then packed into two words (flags, in-group ranks).
#pragma unroll 1
        for (int L0 = S.lmin; L0 < h; L0 += 4) {
            uint32_t fl[4], pr[4];
            {
                uint4 a[4], bw[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    a[j] = bw[j] = make_uint4(0u, 0u, 0u, 0u);
                    const int L = L0 + j;
                    if (valid && L < h) {
                        const LevelDesc lv = S.lev[L];
                        ldg256(S.flagrec + flag_index(S, lv.pc_base + (uint32_t)((v >> L) * lv.UL + (u >> L)) * 3u, fg) + 2, a[j], bw[j]);
                    }
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t resw[3] = {bw[j].x, bw[j].y, a[j].x}, prdw[3] = {bw[j].z, bw[j].w, a[j].z};
                    fl[j] = pr[j] = 0u;
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        fl[j] |= ((resw[c] & bit) ? 1u << c : 0u) | ((prdw[c] & bit) ? 8u << c : 0u) | ((uint32_t)__popc(resw[c] & (bit - 1u)) << (8 + 5 * c));
                        pr[j] |= (uint32_t)__popc(prdw[c] & (bit - 1u)) << (5 * c);
                    }
                }
            }
#pragma unroll 1  // (the drains are large: one copy of them)
            for (int j = 0; j < 4; ++j) {
                const int L = L0 + j;
                if (L < h) {  // warp-uniform
                const uint32_t flj = j == 0 ? fl[0] : j == 1 ? fl[1] : j == 2 ? fl[2] : fl[3];
                const uint32_t prj = j == 0 ? pr[0] : j == 1 ? pr[1] : j == 2 ? pr[2] : pr[3];
                const int pu = u >> L, pv = v >> L;
                const LevelDesc lv = S.lev[L];
                const uint32_t base = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
                const uint32_t rbase = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
                const bool predictive = ((pu | pv) & 1) != 0;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const uint32_t dest = (uint32_t)(lane * 4 + c);
                    const bool res = (flj >> c) & 1u;
                    push(q.vq, vcnt, res, make_uint4(base + (uint32_t)c, fg, kin | (((flj >> (8 + 5 * c)) & 31u) << 8) | (dest << 24), 0u), lane_lt);
                    if (vcnt >= 32) drain_v<kMode>(S, q, vcnt, 32, lane, lut);
                    const bool pred = predictive && ((flj >> (3 + c)) & 1u);
                    push(q.mq, mcnt, pred, make_uint4(base + (uint32_t)c, fg, rbase + (uint32_t)c, dest | (((prj >> (5 * c)) & 31u) << 8)), lane_lt);
                    if (mcnt >= 32) {
                        drain_m<kMode, kSubpel, kCs>(S, q, mcnt, vcnt, 32, lane, lane_lt, lut);
                        if (vcnt >= 32) drain_v<kMode>(S, q, vcnt, 32, lane, lut);
                    }
                }
                }
            }
        }
    } else {
#pragma unroll 1
    for (int L = S.lmin; L < h; ++L) {
        const int pu = u >> L, pv = v >> L;
        const LevelDesc lv = S.lev[L];
        const uint32_t base = lv.pc_base + (uint32_t)(pv * lv.UL + pu) * 3u;
        const uint32_t rbase = lv.pc_base + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1)) * 3u;
        const bool predictive = ((pu | pv) & 1) != 0;
        // S4: the three channels' descriptors and flag records, six independent loads
        uint4 d[3], fr[3];
        // S4: the three channels' descriptors and their flag records; the records share one 64-byte slot: a 256-bit
        // load (Y, Co) and a 128-bit load (Cg)
#pragma unroll
        for (int c = 0; c < 3; ++c) d[c] = fr[c] = make_uint4(0u, 0u, 0u, 0u);
        if (valid) {
            const uint4 *slot = S.flagrec + flag_index(S, base, fg);
            if (kCs) {  // the chroma records of the plane's slot of group fg_c
                const uint4 *slot_c = S.flagrec + flag_index(S, base, fg_c);
                fr[0] = ldg(slot);
                fr[1] = ldg(slot_c + 1);
                fr[2] = ldg(slot_c + 2);
            } else {
                ldg256(slot, fr[0], fr[1]);
                fr[2] = ldg(slot + 2);
            }
#pragma unroll
            for (int c = 0; c < 3; ++c) d[c] = ldg(S.pc + base + c);
        }
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const uint32_t dest = (uint32_t)(lane * 4 + c);
            const uint32_t bit = c ? bit_c : bit0, kin = c ? kin_c : kin0;
            const bool res = (fr[c].x & bit) != 0u;
            const uint32_t rank = fr[c].y + (uint32_t)__popc(fr[c].x & (bit - 1u));
            push(q.vq, vcnt, res, make_uint4(d[c].y, (rank << (2 * S.logB)) + kin, (d[c].w & 0x3FFFFFu) | (dest << 24), 0u), lane_lt);
            if (vcnt >= 32) drain_v<kMode>(S, q, vcnt, 32, lane, lut);
            const bool pred = predictive && (fr[c].z & bit) != 0u;
            const uint32_t mi = fr[c].w + (uint32_t)__popc(fr[c].z & (bit - 1u));
            push(q.mq, mcnt, pred, make_uint4(d[c].z, mi, rbase + (uint32_t)c, dest), lane_lt);
            if (mcnt >= 32) {
                drain_m<kMode, kSubpel, kCs>(S, q, mcnt, vcnt, 32, lane, lane_lt, lut);
                if (vcnt >= 32) drain_v<kMode>(S, q, vcnt, 32, lane, lut);
            }
        }
    
    }
    }
    if (mcnt > 0) drain_m<kMode, kSubpel, kCs>(S, q, mcnt, vcnt, mcnt, lane, lane_lt, lut);
    if (vcnt >= 32) drain_v<kMode>(S, q, vcnt, 32, lane, lut);
    if (vcnt > 0) drain_v<kMode>(S, q, vcnt, vcnt, lane, lut);
    __syncwarp();

    // S8: inverse YCoCg-R + clamp, then the warp's 96 bytes as 24 coalesced words
    uint32_t rgb = 0u;
    if (valid) {
        const int acc[3] = {q.acc[lane * 4 + 0], q.acc[lane * 4 + 1], q.acc[lane * 4 + 2]};
        rgb = ycocg_to_rgb8(acc);
    }
    const long long wbase = i - lane;
    uint8_t *o = out + 3 * wbase;
    if (out_aligned && wbase + 32 <= n) {
        uint32_t *stage = reinterpret_cast<uint32_t *>(q.vq);  // the warp's 96 output bytes (its stacks are empty)
        uint8_t *sb = reinterpret_cast<uint8_t *>(stage);
        sb[3 * lane + 0] = (uint8_t)(rgb & 0xFF);
        sb[3 * lane + 1] = (uint8_t)((rgb >> 8) & 0xFF);
        sb[3 * lane + 2] = (uint8_t)((rgb >> 16) & 0xFF);
        __syncwarp();
#ifdef HMLFC_DECODE_CS
        if (lane < 24) __stcs(reinterpret_cast<uint32_t *>(o) + lane, stage[lane]);
#else
        if (lane < 24) reinterpret_cast<uint32_t *>(o)[lane] = stage[lane];
#endif
    } else if (present) {
        o[3 * lane + 0] = (uint8_t)(rgb & 0xFF);
        o[3 * lane + 1] = (uint8_t)((rgb >> 8) & 0xFF);
        o[3 * lane + 2] = (uint8_t)((rgb >> 16) & 0xFF);
    }
}


// ---------------------------------------------------------------------------------------------------------------
// hmlfc_decode on the block records (hmlfc_device.cuh): a warp walks kSets x 32 coordinates through the levels and shares its task
// stacks between them (kSets = 1 is what runs, see kBrecSets).  kCg: streams in HBM: the random sectors go through the L2 only.
template <bool kCg, int kSets, int kMinBlocks>
__global__ void __launch_bounds__(kThreads, kMinBlocks)
decode_brec_kernel(const DevStream S, const int4 *__restrict__ coords, long long n, uint8_t *__restrict__ out,
                   unsigned long long *oob, int out_aligned)
{
    __shared__ WarpQT<kCap, kSets> wq[kWarps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const uint32_t lane_lt = (1u << lane) - 1u;
    auto &q = wq[warp];
    const int h = S.h;
    // coordinate of set k: the warp's k-th run of 32 consecutive coordinates
    long long idx[kSets];
    int4 c4[kSets];
    bool valid[kSets];
#pragma unroll
    for (int k = 0; k < kSets; ++k) {
        idx[k] = ((long long)blockIdx.x * kWarps + warp) * (kSets * 32) + k * 32 + lane;
        c4[k] = make_int4(0, 0, 0, 0);
        if (idx[k] < n) c4[k] = __ldg(coords + idx[k]);
    }
#pragma unroll
    for (int k = 0; k < kSets; ++k) {
        valid[k] = idx[k] < n && (unsigned)c4[k].x < (unsigned)S.U && (unsigned)c4[k].y < (unsigned)S.V &&
                   (unsigned)c4[k].z < (unsigned)S.Ws && (unsigned)c4[k].w < (unsigned)S.Ht;
        if (idx[k] < n && !valid[k]) atomicAdd(oob, 1ull);
        // S3 root term: one 64-bit load; the cell starts at the top-level RKV sample
        short4 root = make_short4(0, 0, 0, 0);
        if (valid[k])
            root = ldg(S.rkv + ((size_t)((c4[k].y >> h) * S.UH + (c4[k].x >> h)) * (size_t)S.Ht + (size_t)c4[k].w) * (size_t)S.Ws + (size_t)c4[k].z);
        const int cell = k * 32 + lane;
        q.acc[cell * 4 + 0] = root.x;
        q.acc[cell * 4 + 1] = root.y;
        q.acc[cell * 4 + 2] = root.z;
        q.xy[cell] = (uint32_t)c4[k].z | ((uint32_t)c4[k].w << 16);
    }
    int vcnt = 0, mcnt = 0, rcnt = 0;
    // S4 on the block records: per level ONE sector (the slot of the block's group in the level's plane) says what the plane holds for
    // the sample and where; the plane's descriptor (16 bytes, a few hundred KB in all) gives widths and offsets.  The level loop runs
    // one extra round that only flushes (one copy of the flush code).
#pragma unroll 1
    for (int L = S.lmin; L <= h; ++L) {
        const bool flush = L == h;
        if (!flush) {
            const LevelDesc lv = S.lev[L];
            const uint32_t plane0 = umulhi(lv.pc_base, 0xAAAAAAABu) >> 1;  // pc_base / 3
#pragma unroll
            for (int k = 0; k < kSets; ++k) {
                const int pu = c4[k].x >> L, pv = c4[k].y >> L;
                const uint32_t plane = plane0 + (uint32_t)(pv * lv.UL + pu), rplane = plane0 + (uint32_t)((pv & ~1) * lv.UL + (pu & ~1));
                const bool predictive = ((pu | pv) & 1) != 0;
                const int b = valid[k] ? (c4[k].w >> S.logB) * S.nbx + (c4[k].z >> S.logB) : 0;
                const uint32_t kin = (uint32_t)(((c4[k].w & (S.B - 1)) << S.logB) + (c4[k].z & (S.B - 1)));
                uint4 sa = make_uint4(0u, 0u, 0u, 0u), sb = sa, pb = sa;
                if (valid[k]) {
                    const uint4 *slot = S.bslot + ((size_t)plane * (size_t)S.fgroups + (size_t)(b >> 5)) * 2u;
                    if (kCg) ldcg256(slot, sa, sb); else ldg256(slot, sa, sb);
                    pb = ldg(S.pb + plane);
                }
                const BrecPos r = brec_locate(S, sa, sb, 1u << (b & 31), pb);
                const unsigned long long vpos = r.bit + brec_sample_offset(r, pb, kin);
                const uint32_t cell = (uint32_t)(k * 32 + lane);
                push(q.vq, vcnt, r.res != 0u, make_uint4((uint32_t)(vpos >> 5), value_what((uint32_t)vpos & 31u, r.res, r.res, 0u, pb, cell), pb.z, pb.w), lane_lt);
                push(q.mq, mcnt, predictive && r.pred != 0u,
                     make_uint4((uint32_t)(r.bit >> 5), ((uint32_t)r.bit & 31u) | (r.pred << 5) | (cell << 8), rplane, 0u), lane_lt);
                // the usual order, inline (4% faster than going through the loop below)
                if (vcnt >= 32) drain_values_brec<kCg>(S, q, vcnt, 32, lane);
                if (mcnt >= 32) drain_motion_brec<kCg>(S, q, mcnt, rcnt, vcnt, 32, lane, lane_lt);
            }
            continue;
        }
#pragma unroll 1
        while (true) {
            const int which = vcnt >= 32 ? 0 : rcnt >= 32 ? 1 : mcnt > 0 ? 2 : rcnt > 0 ? 1 : vcnt > 0 ? 0 : -1;
            if (which < 0) break;
            if (which == 0) drain_values_brec<kCg>(S, q, vcnt, min(vcnt, 32), lane);
            else if (which == 1) drain_lookups_brec<kCg>(S, q, rcnt, vcnt, min(rcnt, 32), lane, lane_lt);
            else drain_motion_brec<kCg>(S, q, mcnt, rcnt, vcnt, min(mcnt, 32), lane, lane_lt);
        }
    }
    __syncwarp();
    // S8: inverse YCoCg-R + clamp, then each set's 96 bytes as 24 coalesced words (staged in the empty value stack)
    uint32_t *stage = reinterpret_cast<uint32_t *>(q.vq);
#pragma unroll
    for (int k = 0; k < kSets; ++k) {
        uint32_t rgb = 0u;
        if (valid[k]) {
            const int cell = k * 32 + lane;
            const int acc[3] = {q.acc[cell * 4 + 0], q.acc[cell * 4 + 1], q.acc[cell * 4 + 2]};
            rgb = ycocg_to_rgb8(acc);
        }
        const long long wbase = idx[k] - lane;
        uint8_t *o = out + 3 * wbase;
        if (out_aligned && wbase + 32 <= n) {
            uint8_t *sb = reinterpret_cast<uint8_t *>(stage + 24 * k);
            sb[3 * lane + 0] = (uint8_t)(rgb & 0xFF);
            sb[3 * lane + 1] = (uint8_t)((rgb >> 8) & 0xFF);
            sb[3 * lane + 2] = (uint8_t)((rgb >> 16) & 0xFF);
            __syncwarp();
            if (lane < 24) reinterpret_cast<uint32_t *>(o)[lane] = stage[24 * k + lane];
        } else if (idx[k] < n) {
            o[3 * lane + 0] = (uint8_t)(rgb & 0xFF);
            o[3 * lane + 1] = (uint8_t)((rgb >> 8) & 0xFF);
            o[3 * lane + 2] = (uint8_t)((rgb >> 16) & 0xFF);
        }
    }
}

}  // namespace

// The block-record kernel lives on L1 hits (plane descriptors, neighbouring fields) as much as on occupancy: 6 CTAs per SM leave 60 KB of
// L1, 5 leave 92 KB.  Measured (G px/s, 6 / 5 CTAs): cfg2 (stream in the L2) 14.8 / 14.4, cfg4 (in HBM) 6.0 / 7.3 -- instantiation 3 is the
// kernel with a shared-memory carve-out that fits 5 CTAs, used for streams the L2 does not hold.
cudaError_t configure_decode_queue()
{
    return cudaFuncSetAttribute(decode_brec_kernel<true, kBrecSets, 5>, cudaFuncAttributePreferredSharedMemoryCarveout, 65);
}

cudaError_t launch_decode_queue(const DevStream &S, const int32_t *d_coords, int64_t n, uint8_t *d_out,
                                unsigned long long *d_oob, cudaStream_t st, int *n_launches, int mode)
{
    if (n == 0) return cudaSuccess;
    if (S.Ws > 65536 || S.Ht > 65536) return cudaErrorInvalidValue;  // s | t << 16 packing
    const long long blocks = (n + kThreads - 1) / kThreads;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0) ? 1 : 0;
    // mode: 0 eager, 1 lazy, 2 block records (needs S.brec); < 0: chosen here
    if (mode < 0) mode = S.brec ? 2 : (S.l2_resident ? 1 : 0);
    if (S.sp || S.cs) mode = 0;  // half-pel / chroma-subsampled streams: the eager form has their instantiations (and they have no block records)
    if (mode == 2 && !S.brec) return cudaErrorInvalidValue;
    const int4 *c4 = reinterpret_cast<const int4 *>(d_coords);
    if (mode == 2) {
        const long long per_cta = (long long)kThreads * kBrecSets, cb = (n + per_cta - 1) / per_cta;
        if (S.l2_resident) decode_brec_kernel<false, kBrecSets, 6><<<(unsigned)cb, kThreads, 0, st>>>(S, c4, (long long)n, d_out, d_oob, aligned);
        else decode_brec_kernel<true, kBrecSets, 5><<<(unsigned)cb, kThreads, 0, st>>>(S, c4, (long long)n, d_out, d_oob, aligned);  // larger L1: configure_decode_queue
    } else if (mode == 1)
        decode_queue_kernel<0, 1><<<(unsigned)blocks, kThreads, 0, st>>>(S, c4, (long long)n, d_out, d_oob, aligned);
    else if (S.cs && S.sp)
        decode_queue_kernel<0, 0, true, true><<<(unsigned)blocks, kThreads, 0, st>>>(S, c4, (long long)n, d_out, d_oob, aligned);
    else if (S.cs)
        decode_queue_kernel<0, 0, false, true><<<(unsigned)blocks, kThreads, 0, st>>>(S, c4, (long long)n, d_out, d_oob, aligned);
    else if (S.sp)
        decode_queue_kernel<0, 0, true><<<(unsigned)blocks, kThreads, 0, st>>>(S, c4, (long long)n, d_out, d_oob, aligned);
    else
        decode_queue_kernel<0, 0><<<(unsigned)blocks, kThreads, 0, st>>>(S, c4, (long long)n, d_out, d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_decode_blocks(const DevStream &S, const int32_t *d_blocks, int64_t n_blocks, uint8_t *d_out, unsigned long long *d_oob,
                                 cudaStream_t st, int *n_launches)
{
    if (n_blocks == 0) return cudaSuccess;
    if (S.Ws > 65536 || S.Ht > 65536) return cudaErrorInvalidValue;
    const long long n = (long long)n_blocks * S.B * S.B;
    const long long blocks = (n + kThreads - 1) / kThreads;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0) ? 1 : 0;
    decode_queue_kernel<2, 0><<<(unsigned)blocks, kThreads, 0, st>>>(S, reinterpret_cast<const int4 *>(d_blocks), n, d_out, d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

cudaError_t launch_decode_views(const DevStream &S, const int32_t *d_views, int64_t n_views, uint8_t *d_out, unsigned long long *d_oob,
                                cudaStream_t st, int *n_launches)
{
    if (n_views == 0) return cudaSuccess;
    if (S.Ws > 65536 || S.Ht > 65536) return cudaErrorInvalidValue;
    const long long n = (long long)n_views * S.Ws * S.Ht;
    const long long blocks = (n + kThreads - 1) / kThreads;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const int aligned = ((reinterpret_cast<uintptr_t>(d_out) & 3u) == 0) ? 1 : 0;
    decode_queue_kernel<1, 0><<<(unsigned)blocks, kThreads, 0, st>>>(S, reinterpret_cast<const int4 *>(d_views), n, d_out, d_oob, aligned);
    if (n_launches) *n_launches += 1;
    return cudaGetLastError();
}

}  // namespace hmlfc
