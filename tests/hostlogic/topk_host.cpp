// Host build of csrc/topk_list.h for tests/test_topk_list.py (plain memory policy).
#include "topk_list.h"

namespace {
struct HostMem {
    template <class T> static T ld(const T* p) { return *p; }
    template <class T> static void st(T* p, T v) { *p = v; }
};
}  // namespace

extern "C" int host_list_insert(int kp, float* Ln, int* Lj, int K, float cn, int cj) {
    if (kp == 8 && K <= 8) kbmod::list_insert<8, HostMem>(Ln, Lj, K, cn, cj);
    else if (kp == 0) kbmod::list_insert<0, HostMem>(Ln, Lj, K, cn, cj);
    else return -1;
    return 0;
}
