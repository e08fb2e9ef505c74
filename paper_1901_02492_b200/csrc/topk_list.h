// topk_list.h -- S6: the per-pixel sorted candidate list (nu descending, ties: smaller velocity
// index first; Eq.27, tie rule DESIGN.md Q15).  Plain functions over a memory policy
// so that the same code runs in the staged kernel (L2 loads/stores on the output planes) and in
// the host-side unit test (tests/test_topk_list.py).
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define KBMOD_HD __host__ __device__ __forceinline__
#else
#define KBMOD_HD inline
#endif

namespace kbmod {

// candidate (cn, cj) ranks before entry (pn, pj)
KBMOD_HD bool better(float cn, int cj, float pn, int pj) { return cn > pn || (cn == pn && cj < pj); }

constexpr int LIST_EMPTY_IDX = 0x7FFFFFFF;     // empty slot = (-inf, LIST_EMPTY_IDX): ranks last

// Sorted insert of (cn, cj) into the list Ln[0..K), Lj[0..K).  KP > 0: K <= KP, the whole list is
// held in registers and written back where it changed (one memory round trip); KP == 0: any K,
// entries are shifted down one by one from the tail.  Mem::ld / Mem::st do the accesses.
template <int KP, class Mem>
KBMOD_HD void list_insert(float* Ln, int* Lj, int K, float cn, int cj) {
    if constexpr (KP > 0) {
        float ln[KP];
        int lj[KP];
#pragma unroll
        for (int e = 0; e < KP; ++e) {
            ln[e] = (e < K) ? Mem::ld(Ln + e) : INFINITY;     // beyond K: never displaced
            lj[e] = (e < K) ? Mem::ld(Lj + e) : -1;
        }
        bool gt[KP];
#pragma unroll
        for (int e = 0; e < KP; ++e) gt[e] = better(cn, cj, ln[e], lj[e]);
        // the list is sorted, so gt is false...false,true...true: slot e takes its upper
        // neighbour if that one is displaced too, else the candidate
#pragma unroll
        for (int e = KP - 1; e >= 0; --e) {
            if (e < K && gt[e]) {
                const bool shift = (e > 0) && gt[e > 0 ? e - 1 : 0];
                Mem::st(Ln + e, shift ? ln[e > 0 ? e - 1 : 0] : cn);
                Mem::st(Lj + e, shift ? lj[e > 0 ? e - 1 : 0] : cj);
            }
        }
    } else {
        if (!better(cn, cj, Mem::ld(Ln + K - 1), Mem::ld(Lj + K - 1))) return;
        int e = K - 1;
        while (e > 0) {
            const float pn = Mem::ld(Ln + e - 1);
            const int pj = Mem::ld(Lj + e - 1);
            if (!better(cn, cj, pn, pj)) break;
            Mem::st(Ln + e, pn);
            Mem::st(Lj + e, pj);
            --e;
        }
        Mem::st(Ln + e, cn);
        Mem::st(Lj + e, cj);
    }
}

}  // namespace kbmod
