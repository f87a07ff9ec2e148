// ccl_unionfind.cuh -- device-side root finding and Algorithm 1, shared by the direct and the
// region-bucketed forms of step (iii).  Product code (no oracle code is included here or includes this).
#pragma once

#include "ccl_common.cuh"

namespace ccl {

// ------------------------------------------------------------------------------------------ root finding
// Walk label[label[...]] to the root, halving the path on the way: every visited site is
// re-pointed at its grandparent.  A shortcut store can only write an ancestor, so it never disconnects anything
// (DESIGN.md "Concurrency").
__device__ __forceinline__ int32_t find_root(int32_t* label, int32_t x)
{
    int32_t p = ld_label(label + x);
    while (p != x) {
        const int32_t gp = ld_label(label + p);
        if (gp == p) return p;
        st_label(label + x, gp);
        x = gp;
        p = ld_label(label + x);
    }
    return x;
}

// The two root walks of Algorithm 1 advanced together: both chains issue their loads in the same
// step, so the dependent-load depth is the longer of the two walks instead of their sum.  Same path halving.
__device__ __forceinline__ void find_roots2(int32_t* label, int32_t& a, int32_t& b)
{
    int32_t pa = ld_label(label + a), pb = ld_label(label + b);        // invariant: pa = a value read from label[a]
    for (;;) {
        const bool wa = pa != a, wb = pb != b;                         // still walking?
        if (!wa && !wb) return;
        const int32_t ga = wa ? ld_label(label + pa) : pa;             // grandparents, both loads in flight together
        const int32_t gb = wb ? ld_label(label + pb) : pb;
        bool la = false, lb = false;
        if (wa) {
            if (ga == pa) a = pa;                                      // pa is a root (and pa == a now)
            else { st_label(label + a, ga); a = ga; la = true; }       // halve: a -> grandparent, move there
        }
        if (wb) {
            if (gb == pb) b = pb;
            else { st_label(label + b, gb); b = gb; lb = true; }
        }
        const int32_t na = la ? ld_label(label + a) : pa;
        const int32_t nb = lb ? ld_label(label + b) : pb;
        pa = na; pb = nb;
    }
}

// Algorithm 1 (reading R3 of its garbled last lines, exit test R4): make sure sites a and b end
// up in one tree.  label_1 is the larger of the two current representatives, label_2 the smaller.
__device__ __forceinline__ void algorithm1(int32_t* label, int32_t a, int32_t b)
{
    int32_t label_1 = a, label_2 = b;
    find_roots2(label, label_1, label_2);
    while (label_1 != label_2) {
        if (label_1 < label_2) { const int32_t t = label_1; label_1 = label_2; label_2 = t; }
        const int32_t label_3 = atomicMin(label + label_1, label_2);
        if (label_3 == label_1 || label_3 == label_2) return;     // linked now / was linked already
        // label_1 was not a root any more.  If label_3 > label_2 the link label_1 -> label_3 has just been
        // replaced by label_1 -> label_2, so label_3 must be joined to label_2; if label_3 < label_2 nothing was
        // written and label_1 hangs under label_3, which must be joined to label_2.  Either way the pair to join
        // is (label_3, label_2); walk both up to their roots before the next atomic.
        label_1 = label_3;
        find_roots2(label, label_1, label_2);
    }
}

}  // namespace ccl
