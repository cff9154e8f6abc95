// tcw_median.cuh -- exact running median over a sliding window, amortised O(1) per slide (sm_100a).
//
// tcw_prepare's noise floor is m_j[k] = median of P_j[k-h .. k+h] (reading Q24).  A thread walks
// a run of consecutive bins.  Re-counting the window for every bin costs ~W compares per bin; here the
// thread keeps, in registers,
//   m              the current median VALUE (the rank-h order statistic of the window, ranks from 0),
//   c_less, c_eq   how many window elements are < m and == m   (invariant: c_less <= h < c_less + c_eq),
//   lo[], hi[]     the window elements just below / just above m, sorted away from m, COMPLETE inside
//                  their bounds: every window element x with lo_bound < x < m is in lo[] (with its
//                  multiplicity), every x with m < x < hi_bound is in hi[].
// A slide removes one element and inserts one: both touch the two counters and at most one list.  When
// the invariant breaks the median moves by one distinct value, which the lists supply (the old median's
// copies move to the other list).  Only when the needed list is empty is the window re-scanned (for the
// MED_K nearest elements on that side), about once in MED_K^2 slides for random data.  Values compare as
// floats (P >= 0, no NaN: |X|^2 of finite data); equal values are handled by multiplicity, so the result
// is the exact order statistic whatever the ties.
#pragma once

#ifndef TCW_HD
#ifdef __CUDACC__
#define TCW_HD __host__ __device__ __forceinline__
#else
#define TCW_HD inline
#endif
#endif

namespace tcw {

constexpr int MED_K = 8;
#define TCW_MED_INF __builtin_huge_valf()

struct MedianState {
    float m;
    int c_less, c_eq;
    float lo[MED_K], hi[MED_K];     // lo descending (lo[0] nearest below m), hi ascending (hi[0] nearest above m)
    int n_lo, n_hi;
    float lo_bound, hi_bound;       // elements <= lo_bound / >= hi_bound are not tracked
};

// sorted insert of v into a "nearest first" list; NEAR(a, b) is true when a is nearer to m than b
template <bool BELOW>
TCW_HD void med_insert(float (&l)[MED_K], int &n, float &bound, float v)
{
    // entries nearer than v stay, v goes in front of the first entry that is not nearer
    float carry = v;
    bool placed = false;
#pragma unroll
    for (int i = 0; i < MED_K; ++i) {
        if (i < n) {
            const bool keep = placed ? false : (BELOW ? l[i] >= carry : l[i] <= carry);
            if (!keep) { const float t = l[i]; l[i] = carry; carry = t; placed = true; }
        }
    }
    if (n < MED_K) { l[n] = carry; ++n; return; }
    // overflow: `carry` is the farthest element.  It becomes the bound, and the list may keep no element
    // equal to the bound (copies of it outside the list are unknown).
    bound = carry;
    while (n > 0 && l[n - 1] == bound) --n;
}

// remove one copy of v (known to be inside the list's bounds, hence present)
TCW_HD void med_remove(float (&l)[MED_K], int &n, float v)
{
    bool found = false;
#pragma unroll
    for (int i = 0; i < MED_K; ++i) {
        if (i < n) {
            if (!found && l[i] == v) found = true;
            if (found && i + 1 < MED_K) l[i] = l[i + 1];
        }
    }
    if (found) --n;
}

// exact rank-h element of win[0..W) by a bitwise binary search on the float bits (all values >= 0)
template <typename Load>
TCW_HD float med_select(Load win, int W, int h)
{
    unsigned int key = 0;
    for (int bit = 30; bit >= 0; --bit) {
        const unsigned int cand = key | (1u << bit);
        int c = 0;
        for (int q = 0; q < W; ++q) c += win.bits(q) < cand;
        if (c <= h) key = cand;
    }
    return win.from_bits(key);
}

// (re)build the state for the window win[0..W): median by selection, counters by one scan, lists empty
template <typename Load>
TCW_HD void med_init(MedianState &s, Load win, int W, int h)
{
    s.m = med_select(win, W, h);
    s.c_less = s.c_eq = 0;
    for (int q = 0; q < W; ++q) {
        const float x = win.value(q);
        s.c_less += x < s.m;
        s.c_eq += x == s.m;
    }
    s.n_lo = s.n_hi = 0;
    s.lo_bound = s.hi_bound = s.m;      // nothing known on either side
}

// collect the MED_K nearest window elements below (BELOW) or above m into the list
template <bool BELOW, typename Load>
TCW_HD void med_rescan(MedianState &s, Load win, int W)
{
    float (&l)[MED_K] = BELOW ? s.lo : s.hi;
    int &n = BELOW ? s.n_lo : s.n_hi;
    float &bound = BELOW ? s.lo_bound : s.hi_bound;
    n = 0;
    bound = BELOW ? -TCW_MED_INF : TCW_MED_INF;
    for (int q = 0; q < W; ++q) {
        const float x = win.value(q);
        if (BELOW ? (x < s.m && x > bound) : (x > s.m && x < bound)) med_insert<BELOW>(l, n, bound, x);
    }
}

// the window slid by one: `out` left, `in` entered; `win` views the NEW window.  Returns the new median.
template <typename Load>
TCW_HD float med_slide(MedianState &s, Load win, int W, int h, float out, float in)
{
    if (out < s.m) { --s.c_less; if (out > s.lo_bound) med_remove(s.lo, s.n_lo, out); }
    else if (out == s.m) --s.c_eq;
    else if (out < s.hi_bound) med_remove(s.hi, s.n_hi, out);
    if (in < s.m) { ++s.c_less; if (in > s.lo_bound) med_insert<true>(s.lo, s.n_lo, s.lo_bound, in); }
    else if (in == s.m) ++s.c_eq;
    else if (in < s.hi_bound) med_insert<false>(s.hi, s.n_hi, s.hi_bound, in);

    if (s.c_less > h) {
        // the median moves down to the largest element below m
        if (s.n_lo == 0) {
            med_rescan<true>(s, win, W);
            if (s.n_lo == 0) { med_init(s, win, W, h); return s.m; }     // MED_K or more copies of one value: start over
        }
        const float v = s.lo[0];
        int e = 0;
#pragma unroll
        for (int i = 0; i < MED_K; ++i) e += (i < s.n_lo && s.lo[i] == v);
        for (int c = 0; c < s.c_eq; ++c) {                               // the old median's copies are now the nearest above
            if (!(s.m < s.hi_bound)) break;
            med_insert<false>(s.hi, s.n_hi, s.hi_bound, s.m);
        }
        for (int c = 0; c < e; ++c) med_remove(s.lo, s.n_lo, v);
        s.c_less -= e;
        s.c_eq = e;
        s.m = v;
    } else if (s.c_less + s.c_eq <= h) {
        // the median moves up to the smallest element above m
        if (s.n_hi == 0) {
            med_rescan<false>(s, win, W);
            if (s.n_hi == 0) { med_init(s, win, W, h); return s.m; }
        }
        const float v = s.hi[0];
        int e = 0;
#pragma unroll
        for (int i = 0; i < MED_K; ++i) e += (i < s.n_hi && s.hi[i] == v);
        for (int c = 0; c < s.c_eq; ++c) {
            if (!(s.m > s.lo_bound)) break;
            med_insert<true>(s.lo, s.n_lo, s.lo_bound, s.m);
        }
        for (int c = 0; c < e; ++c) med_remove(s.hi, s.n_hi, v);
        s.c_less += s.c_eq;
        s.c_eq = e;
        s.m = v;
    }
    return s.m;
}

}  // namespace tcw
