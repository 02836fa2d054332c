// xs1024.cuh -- the paper's XORShift1024 update (eq.(8); (a,b,c) = (329,347,344),
// PAPER.md:177; Listing 1) for an instance spread over P = 32/K lanes of a
// warp, K consecutive words per lane (word 0 = most significant, R-D1).
//
//   K = 1  : the paper's layout, one word per thread, 32 threads per instance; the exchange
//            is a warp shuffle instead of the paper's padded volatile shared array
//            (footnote 3, anticipates it).  6 shuffles per draw.
//   K = 2..16: the instance lives in 16..2 lanes; a lane needs only K+1 foreign words per
//            phase, i.e. 3(K+1)/K shuffles per draw, and a warp hosts K instances.
//   K = 32 : the whole instance in the registers of one thread; no exchange at all.
// The three phases, with s_j = 0 outside [0,31] (the paper's zero padding)
// and every phase reading pre-phase words:
//   A (X ^= X << 329): s_i ^= (s_{i+10} <<  9) | (s_{i+11} >> 23)
//   B (X ^= X >> 347): s_i ^= (s_{i-10} >> 27) | (s_{i-11} <<  5)
//   C (X ^= X << 344): s_i ^= (s_{i+10} << 24) | (s_{i+11} >>  8)
// All 32 lanes of the warp must call (full-mask shuffles of width P).
// Product code (sm_100a); shares nothing with oracle/.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace rngb200 {

// Lane masks of the zero padding.  With K words per lane every foreign word of a phase comes
// from one of two lanes, D = 10/K or D+1 lanes away (K = 32: none).  A mask is all-ones when
// that lane belongs to the instance; it is made opaque to the compiler so that it stays an
// AND operand that folds into the LOP3 of the xor (instead of one SEL per shuffled word).
// A word whose two sources sit in DIFFERENT lanes (D and D+1 away; one such word per phase, every word for K = 1)
// is masked AFTER the funnel shift: the shifted word takes its upper bits from one source and its lower bits
// from the other, so "source a masked by ma, source b by mb" equals the shift of the unmasked pair ANDed with
// the same shift of (ma, mb) -- a per-lane constant per phase (mix[]), which again folds into the xor's LOP3.
template <int K>
struct XsMasks {
    uint32_t down[2], up[2]; // [0]: D lanes away, [1]: D+1 lanes away
    uint32_t mix[3];         // phases A, B, C: the shifted pair of masks for a word with sources in both lanes
    __device__ __forceinline__ void init(int p)
    {
        constexpr int P = 32 / K, D = 10 / K;
#pragma unroll
        for (int i = 0; i < 2; i++) {
            down[i] = (p + D + i < P) ? 0xffffffffu : 0u;
            up[i] = (p >= D + i) ? 0xffffffffu : 0u;
        }
        mix[0] = __funnelshift_l(down[1], down[0], 9);
        mix[1] = __funnelshift_r(up[0], up[1], 27);
        mix[2] = __funnelshift_l(down[1], down[0], 24);
        if (P > 1) {
#pragma unroll
            for (int i = 0; i < 2; i++) {
                asm volatile("" : "+r"(down[i]));
                asm volatile("" : "+r"(up[i]));
            }
#pragma unroll
            for (int i = 0; i < 3; i++) asm volatile("" : "+r"(mix[i]));
        }
    }
};

// s_i ^= (s_{i+10} << SH) | (s_{i+11} >> (32-SH)) for the K words i = K p + j of this lane
template <int K, int SH, int PH>
__device__ __forceinline__ void xs1024_phase_left(uint32_t (&w)[K], const XsMasks<K> &m)
{
    constexpr int P = 32 / K;
    constexpr unsigned FULL = 0xffffffffu;
    uint32_t nb[K + 1]; // nb[t] = s_{K p + 10 + t} (unmasked where the source lane is out of range)
#pragma unroll
    for (int t = 0; t <= K; t++) {
        const int e = 10 + t, dl = e / K, sl = e % K; // source: lane p + dl, slot sl
        if (dl == 0) nb[t] = w[sl];
        else if (dl >= P) nb[t] = 0u;
        else nb[t] = __shfl_down_sync(FULL, w[sl], dl, P);
    }
#pragma unroll
    for (int j = 0; j < K; j++) { // ascending: in-place safe when the sources are own registers
        const int dh = (10 + j) / K, dlo = (11 + j) / K;
        uint32_t hi = nb[j], lo = nb[j + 1];
        constexpr int D = 10 / K;
        const uint32_t mh = dh == 0 ? 0xffffffffu : dh >= P ? 0u : m.down[dh - D];
        const uint32_t ml = dlo == 0 ? 0xffffffffu : dlo >= P ? 0u : m.down[dlo - D];
        if (dh == dlo) {
            w[j] ^= __funnelshift_l(lo, hi, SH) & mh; // one LOP3: xor with a masked operand
        } else if (dh == D && dlo == D + 1) {
            w[j] ^= __funnelshift_l(lo, hi, SH) & m.mix[PH];
        } else {
            w[j] ^= __funnelshift_l(lo & ml, hi & mh, SH);
        }
    }
}

// s_i ^= (s_{i-10} >> SH) | (s_{i-11} << (32-SH))
template <int K, int SH, int PH>
__device__ __forceinline__ void xs1024_phase_right(uint32_t (&w)[K], const XsMasks<K> &m)
{
    constexpr int P = 32 / K;
    constexpr unsigned FULL = 0xffffffffu;
    uint32_t nb[K + 1]; // nb[t] = s_{K p - 11 + t}
#pragma unroll
    for (int t = 0; t <= K; t++) {
        const int e = t - 11;
        const int du = e >= 0 ? 0 : (-e + K - 1) / K; // lanes up
        const int sl = e + du * K;
        if (du == 0) nb[t] = w[sl];
        else if (du >= P) nb[t] = 0u;
        else nb[t] = __shfl_up_sync(FULL, w[sl], du, P);
    }
#pragma unroll
    for (int j = K - 1; j >= 0; j--) { // descending: in-place safe
        const int eh = j - 11, el = j - 10;
        const int duh = eh >= 0 ? 0 : (-eh + K - 1) / K, dul = el >= 0 ? 0 : (-el + K - 1) / K;
        uint32_t hi = nb[j], lo = nb[j + 1];
        constexpr int D = 10 / K;
        const uint32_t mh = duh == 0 ? 0xffffffffu : duh >= P ? 0u : m.up[duh - D];
        const uint32_t ml = dul == 0 ? 0xffffffffu : dul >= P ? 0u : m.up[dul - D];
        if (duh == dul) {
            w[j] ^= __funnelshift_r(lo, hi, SH) & mh;
        } else if (dul == D && duh == D + 1) {
            w[j] ^= __funnelshift_r(lo, hi, SH) & m.mix[PH];
        } else {
            w[j] ^= __funnelshift_r(lo & ml, hi & mh, SH);
        }
    }
}

// one update of the instance; m = XsMasks of this lane's index within its instance (lane % P)
template <int K>
__device__ __forceinline__ void xs1024_update_k(uint32_t (&w)[K], const XsMasks<K> &m)
{
    xs1024_phase_left<K, 9, 0>(w, m);   // 329 = 10*32 +  9
    xs1024_phase_right<K, 27, 1>(w, m); // 347 = 10*32 + 27
    xs1024_phase_left<K, 24, 2>(w, m);  // 344 = 10*32 + 24
}

// K consecutive 32-bit words, 4K-byte aligned
template <int K>
__device__ __forceinline__ void load_words(const uint32_t *__restrict__ src, uint32_t (&w)[K])
{
    if constexpr (K % 4 == 0) {
#pragma unroll
        for (int q = 0; q < K / 4; q++) {
            const uint4 v = reinterpret_cast<const uint4 *>(src)[q];
            w[4 * q] = v.x, w[4 * q + 1] = v.y, w[4 * q + 2] = v.z, w[4 * q + 3] = v.w;
        }
    } else if constexpr (K == 2) {
        const uint2 v = *reinterpret_cast<const uint2 *>(src);
        w[0] = v.x, w[1] = v.y;
    } else {
#pragma unroll
        for (int q = 0; q < K; q++) w[q] = src[q];
    }
}
template <int K>
__device__ __forceinline__ void store_words(uint32_t *__restrict__ dst, const uint32_t (&w)[K])
{
    if constexpr (K % 4 == 0) {
#pragma unroll
        for (int q = 0; q < K / 4; q++)
            reinterpret_cast<uint4 *>(dst)[q] = make_uint4(w[4 * q], w[4 * q + 1], w[4 * q + 2], w[4 * q + 3]);
    } else if constexpr (K == 2) {
        *reinterpret_cast<uint2 *>(dst) = make_uint2(w[0], w[1]);
    } else {
#pragma unroll
        for (int q = 0; q < K; q++) dst[q] = w[q];
    }
}

} // namespace rngb200
