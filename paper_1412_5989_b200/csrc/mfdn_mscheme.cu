// H1-H6: the coupled-JT -> M-scheme transformation kernels and their launchers.
//
// What one request computes:
//   3-body  v = sign * sum_J sum_{J12} cb(J12,J) * sum_{J12'} ck(J12',J) * sum_{s<5} w[s] * slab[J,J12,J12'][s]
//           cb(J12,J) = <ja ma jb mb|J12 M12> <J12 M12 jc mc|J M>,  ck likewise for the ket,
//           w[s] = isospin weights of the five (T12,T12',T) combinations ("the isospin
//           coupling coefficients are precalculated with several conditionals, and the isospin loops are
//           unrolled into a single weighted summation. The core ... three nested loops over coupled
//           angular momentum values").
//   2-body  v = sign * sqrt((1+d_ab)(1+d_cd)) * sum_J cg_b(J) cg_k(J) * (w0*cell[J][0] + w1*cell[J][1])
// The slab of a (bra tuple, ket tuple) group is stored in exactly this loop order (A2).
//
// Pipeline of one call:
//   k_keys        H1  decode, selection S1-S7 -> mask, canonicalise -> 64-bit record; histogram of the group keys
//   k_scan_*      H2  exclusive scan of the histogram -> bucket bounds
//   k_tscan_*, k_tiles2, k_part<1>, k_part<2>   H2  records -> bucket order by a two-pass partition through shared
//                 memory (skipped if MFDN_PRESORTED)
//   k_items3      H3  one-group work items from the bucket bounds (3-body); groups of <= 16 records on a second list
//   k_transform3  H3-H5  block per item: staged isospin-combined slab, records ordered by M, paired channel sums
//   k_transform3_small   warp per small group, direct sums in the same operation order
//   k_transform2  H3-H5  2-body: warp per 32 records of the group-ordered stream
//   k_back<2>, k_back<1>   H6  values from bucket order back to request order, the same two passes in reverse
//                 (skipped if MFDN_PRESORTED)
//   k_mscheme_naive      MFDN_FORCE_NAIVE: the paper's design, thread per request in request order
#include <algorithm>
#include <chrono>
#include <cstdio>
#include <thread>

#include "mfdn_internal.cuh"

using namespace mfdn;

namespace {

// ------------------------------------------------------------------------------- H1 decode
struct Side3 {
    int tup;       // tuple id or -1
    int ima, imb, imc;
    int tz;        // ta<<2 | tb<<1 | tc
    int twoM, twoMT, par;
    int sign;      // +1 / -1
    bool distinct;
};

__device__ __forceinline__ void cswap(uint32_t& ka, uint32_t& kb, uint32_t& ra, uint32_t& rb, int& sign)
{
    if (ka > kb) {
        uint32_t t = ka; ka = kb; kb = t;
        t = ra; ra = rb; rb = t;
        sign = -sign;
    }
}

// canonicalise three particles: stable sort by (orbital, SPS) ascending, sign of the permutation
template <bool SMEM>
__device__ __forceinline__ Side3 decode3(const Tables& T, const uint32_t* sps, const int2* ab, int s0, int s1, int s2)
{
    Side3 S;
    uint32_t r0 = SMEM ? sps[s0] : __ldg(sps + s0), r1 = SMEM ? sps[s1] : __ldg(sps + s1), r2 = SMEM ? sps[s2] : __ldg(sps + s2);
    uint32_t k0 = (rec_orb(r0) << 16) | s0, k1 = (rec_orb(r1) << 16) | s1, k2 = (rec_orb(r2) << 16) | s2;
    S.distinct = (s0 != s1) && (s0 != s2) && (s1 != s2);
    S.sign = 1;
    cswap(k0, k1, r0, r1, S.sign);
    cswap(k1, k2, r1, r2, S.sign);
    cswap(k0, k1, r0, r1, S.sign);
    int a = rec_orb(r0), b = rec_orb(r1), c = rec_orb(r2);
    if (ab) {   // tuples of a fixed (a, b) are consecutive and their c's form a dense range: {first tuple, cmin | count<<16}
        const int2 e = ab[a * T.n_orb + b];
        const int d = c - (e.y & 0xFFFF);
        S.tup = (e.x >= 0 && (unsigned)d < (unsigned)(e.y >> 16)) ? e.x + d : -1;
    } else {
        S.tup = __ldg(T.tuple_id3 + (a * T.n_orb + b) * T.n_orb + c);
    }
    S.ima = rec_im(r0); S.imb = rec_im(r1); S.imc = rec_im(r2);
    S.tz = (rec_tz(r0) << 2) | (rec_tz(r1) << 1) | rec_tz(r2);
    const uint32_t sum = (r0 >> 10) + (r1 >> 10) + (r2 >> 10);   // every field summed over the three particles at once
    S.twoM = 2 * sum_im(sum) - sum_twoj(sum);
    S.twoMT = 2 * sum_tz(sum) - 3;
    S.par = sum_lpar(sum) & 1;
    return S;
}

// The same from the SPS records as k_keys3s keeps them in shared memory (at most 64 orbitals, 2048 SPS):
//   [26,32) orbital  [15,26) SPS index  [14] l & 1  [12,14) tz bit  [6,12) 2j  [0,6) im
// Sorted as unsigned words they are in (orbital, SPS) order, so the canonical order is min / middle / max (no compare-and-swap
// network with payloads), the sign is the parity of the three pairwise inversions, and the low 15 bits of p0 + p1 + p2 are the
// packed sums of im, 2j, tz and l over the three particles (every sum fits its field: 3 * 21 <= 63).
__host__ __device__ inline uint32_t sps_pack_sorted(uint32_t r, int s)
{
    return ((uint32_t)rec_orb(r) << 26) | ((uint32_t)s << 15) | ((uint32_t)rec_lpar(r) << 14) | ((uint32_t)rec_tz(r) << 12) |
           ((uint32_t)rec_twoj(r) << 6) | (uint32_t)rec_im(r);
}
__device__ __forceinline__ Side3 decode3s(const Tables& T, const uint32_t* sps, const int2* ab, int s0, int s1, int s2)
{
    Side3 S;
    const uint32_t p0 = sps[s0], p1 = sps[s1], p2 = sps[s2], tot = p0 + p1 + p2;
    const uint32_t lo = min(p0, min(p1, p2)), hi = max(p0, max(p1, p2)), mid = tot - lo - hi;
    S.distinct = lo != mid && mid != hi;
    S.sign = ((p0 > p1) != (p1 > p2)) != (p0 > p2) ? -1 : 1;
    const int a = (int)(lo >> 26), b = (int)(mid >> 26), c = (int)(hi >> 26);
    const int2 e = ab[a * T.n_orb + b];
    const int d = c - (e.y & 0xFFFF);
    S.tup = (e.x >= 0 && (unsigned)d < (unsigned)(e.y >> 16)) ? e.x + d : -1;
    S.ima = (int)(lo & 63u); S.imb = (int)(mid & 63u); S.imc = (int)(hi & 63u);
    S.tz = (int)(((lo >> 10) & 4u) | ((mid >> 11) & 2u) | ((hi >> 12) & 1u));
    S.twoM = 2 * (int)(tot & 63u) - (int)((tot >> 6) & 63u);
    S.twoMT = 2 * (int)((tot >> 12) & 3u) - 3;
    S.par = (int)((tot >> 14) & 1u);
    return S;
}

struct Side2 {
    int tup, ima, imb, tz, twoM, twoMT, par, sign;
    bool distinct;
};

template <bool SMEM>
__device__ __forceinline__ Side2 decode2(const Tables& T, const uint32_t* sps, int s0, int s1, const int32_t* s_tid = nullptr)
{
    Side2 S;
    uint32_t r0 = SMEM ? sps[s0] : __ldg(sps + s0), r1 = SMEM ? sps[s1] : __ldg(sps + s1);
    uint32_t k0 = (rec_orb(r0) << 16) | s0, k1 = (rec_orb(r1) << 16) | s1;
    S.distinct = s0 != s1;
    S.sign = 1;
    cswap(k0, k1, r0, r1, S.sign);
    S.tup = s_tid ? s_tid[rec_orb(r0) * T.n_orb + rec_orb(r1)] : __ldg(T.tuple_id2 + rec_orb(r0) * T.n_orb + rec_orb(r1));
    S.ima = rec_im(r0); S.imb = rec_im(r1);
    S.tz = (rec_tz(r0) << 1) | rec_tz(r1);
    const uint32_t sum = (r0 >> 10) + (r1 >> 10);
    S.twoM = 2 * sum_im(sum) - sum_twoj(sum);
    S.twoMT = 2 * sum_tz(sum) - 2;
    S.par = sum_lpar(sum) & 1;
    return S;
}

__device__ __forceinline__ bool in_range(const Tables& T, const int* s, int k)
{
    bool ok = true;
#pragma unroll
    for (int i = 0; i < 6; i++)
        if (i < k) ok = ok && ((unsigned)s[i] < (unsigned)T.n_sps);
    return ok;
}

// selection rules S1-S6 (integer only)
__device__ __forceinline__ bool select3(const Tables& T, const Side3& B, const Side3& K)
{
    return B.distinct && K.distinct && B.twoM == K.twoM && B.twoMT == K.twoMT && B.par == K.par &&
           B.tup >= 0 && K.tup >= 0;   // S5 is implied by S6: listed tuples are within E3max (checked at upload)
}
__device__ __forceinline__ bool select2(const Side2& B, const Side2& K)
{
    return B.distinct && K.distinct && B.twoM == K.twoM && B.twoMT == K.twoMT && B.par == K.par && B.tup >= 0 &&
           K.tup >= 0;
}

// S7 helper: set of (J,T) channels in which this side has an admissible listed state
template <bool SMEM = false>
__device__ __forceinline__ unsigned long long chanmask3(const unsigned long long* stm, int4 d, int twoM12, int twoMT12)
{
    const int J12min = d.y & 255, J12max = (d.y >> 8) & 255;
    const int lo = max(J12min, (abs(twoM12) + 1) >> 1);   // 2*J12 >= |2*M12|
    if (lo > J12max) return 0ull;
    // stmask3 holds suffix ORs over J12: one 16-byte entry {T12 = 0, T12 = 1} covers all J12 >= lo
    const ulonglong2* p = reinterpret_cast<const ulonglong2*>(stm + d.z + (lo - J12min) * 2);
    const ulonglong2 m = SMEM ? *p : __ldg(p);
    return (twoMT12 == 0 ? m.x : 0ull) | m.y;
}

// S7 for a decoded 3-body request that passed S1-S6: at least one admissible channel term
template <bool SMEM = false>
__device__ __forceinline__ bool mask3(const unsigned long long* stm, const Side3& B, const Side3& K, int4 db, int4 dk)
{
    // no test for a common J range of the two tuples: without one the two channel sets below share no (J, T) bit, because the J of
    // every listed state lies inside its tuple's range (checked at upload).  The test cost 11 instructions per request
    // (pre-sorted call of config 3: 2.005 -> 1.951 ms without it)
    const int ja = db.x & 255, jb = (db.x >> 8) & 255, jd = dk.x & 255, je = (dk.x >> 8) & 255;
    const int twoM12b = 2 * (B.ima + B.imb) - ja - jb, twoM12k = 2 * (K.ima + K.imb) - jd - je;
    const int tzb12 = (B.tz >> 2) + ((B.tz >> 1) & 1) - 1, tzk12 = (K.tz >> 2) + ((K.tz >> 1) & 1) - 1;  // MT12
    unsigned long long mm = chanmask3<SMEM>(stm, db, twoM12b, 2 * tzb12) & chanmask3<SMEM>(stm, dk, twoM12k, 2 * tzk12);
    mm &= ~0ull << (2 * (abs(B.twoM) >> 1));                   // J >= |M|
    if (abs(B.twoMT) == 3) mm &= 0xAAAAAAAAAAAAAAAAull;        // T = 3/2 only
    return mm != 0;
}
// the same from the direct look-up table stm12 (Tables::stm12_3), zb / zk = the tuples' offsets in it
__device__ __forceinline__ bool mask3s(const unsigned long long* stm12, const Side3& B, const Side3& K, int zb, int zk)
{
    const int eb = ((B.tz >> 2) ^ (B.tz >> 1)) & 1, ek = ((K.tz >> 2) ^ (K.tz >> 1)) & 1;   // MT12 == 0: the first two tz bits differ
    unsigned long long mm = stm12[zb + (B.ima + B.imb) * 2 + eb] & stm12[zk + (K.ima + K.imb) * 2 + ek];
    mm &= ~0ull << (2 * (abs(B.twoM) >> 1));                   // J >= |M|
    if (abs(B.twoMT) == 3) mm &= 0xAAAAAAAAAAAAAAAAull;        // T = 3/2 only
    return mm != 0;
}
__device__ __forceinline__ bool mask2(const Side2& B, int4 db, int4 dk)
{
    unsigned long long mb = (unsigned long long)(uint32_t)db.z | ((unsigned long long)(uint32_t)db.w << 32);
    unsigned long long mk = (unsigned long long)(uint32_t)dk.z | ((unsigned long long)(uint32_t)dk.w << 32);
    unsigned long long mm = mb & mk & (~0ull << (2 * ((abs(B.twoM) + 1) >> 1)));   // J >= |M|
    if (B.twoMT != 0) mm &= 0xAAAAAAAAAAAAAAAAull;                                 // T = 1 only
    return mm != 0;
}

// ------------------------------------------------------------------------------- request loads
// u16 (MFDN_REQ_U16): the request array holds 16-bit SPS indices, 12 / 8 bytes per request instead of 24 / 16
__device__ __forceinline__ void load_req3(const int32_t* req, long long r, int s[6], int u16)
{
    if (u16) {
        const uint32_t* p = (const uint32_t*)req + 3 * r;
        const uint32_t a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
        s[0] = a & 0xFFFFu; s[1] = a >> 16; s[2] = b & 0xFFFFu; s[3] = b >> 16; s[4] = c & 0xFFFFu; s[5] = c >> 16;
        return;
    }
    const int2* p = (const int2*)(req + 6 * r);
    int2 a = __ldg(p), b = __ldg(p + 1), c = __ldg(p + 2);
    s[0] = a.x; s[1] = a.y; s[2] = b.x; s[3] = b.y; s[4] = c.x; s[5] = c.y;
}
__device__ __forceinline__ void load_req2(const int32_t* req, long long r, int s[6], int u16)
{
    s[4] = 0; s[5] = 0;
    if (u16) {
        const uint2 a = __ldg((const uint2*)req + r);
        s[0] = a.x & 0xFFFFu; s[1] = a.x >> 16; s[2] = a.y & 0xFFFFu; s[3] = a.y >> 16;
        return;
    }
    int4 a = __ldg((const int4*)(req + 4 * r));
    s[0] = a.x; s[1] = a.y; s[2] = a.z; s[3] = a.w;
}

// one value of an isospin-combined slab from global memory (bin base vwb), either storage width
__device__ __forceinline__ double ldvw_global(const uint32_t* __restrict__ vwb, uint32_t gsize, uint32_t cell, int f32)
{
    if (f32) return (double)__uint_as_float(__ldg(vwb + cell));
    return __hiloint2double((int)__ldg(vwb + gsize + cell), (int)__ldg(vwb + cell));
}

// =============================================================================== naive kernel
// MFDN_FORCE_NAIVE: the paper's design -- one thread per request, in request order, the
// loop nest inside the kernel, every index recomputed per thread.  Kept as the on-device reference.
__device__ __forceinline__ double eval3_naive(const Tables& T, const Side3& B, const Side3& K, int& mask)
{
    mask = 0;
    if (!select3(T, B, K)) return 0.0;
    const uint4 sg = __ldg(T.sgrp3 + (size_t)B.tup * T.n_tup3 + K.tup);
    if (sg.x == NO_SLAB) return 0.0;
    const int4 db = __ldg(T.tdesc3 + B.tup), dk = __ldg(T.tdesc3 + K.tup);
    if (!mask3(T.stmask3, B, K, db, dk)) return 0.0;
    mask = 1;
    const int ja = db.x & 255, jb = (db.x >> 8) & 255, jc = (db.x >> 16) & 255;
    const int jd = dk.x & 255, je = (dk.x >> 8) & 255, jf = (dk.x >> 16) & 255;
    const int twoM12b = 2 * (B.ima + B.imb) - ja - jb, twoM12k = 2 * (K.ima + K.imb) - jd - je;
    const int aM = abs(B.twoM);
    const double* ib = T.iso3[B.tz];
    const double* ik = T.iso3[K.tz];
    const double w0 = ib[0] * ik[0], w1 = ib[0] * ik[1], w2 = ib[1] * ik[0], w3 = ib[1] * ik[1], w4 = ib[2] * ik[2];
    const int nj = T.nj;
    const int J12minb = db.y & 255, J12mink = dk.y & 255;
    // CG blocks are [iJ][i1][i2]
    const double* c1b = T.cg1 + __ldg(T.cg1_off + (ja >> 1) * nj + (jb >> 1)) + B.ima * (jb + 1) + B.imb;
    const double* c1k = T.cg1 + __ldg(T.cg1_off + (jd >> 1) * nj + (je >> 1)) + K.ima * (je + 1) + K.imb;
    const int S1b = (ja + 1) * (jb + 1), S1k = (jd + 1) * (je + 1);
    const size_t plane = sg.y;
    const double* row = T.slab3 + (size_t)sg.x * 2;
    const int Jlo = max((db.y >> 16) & 255, (dk.y >> 16) & 255), Jhi = min((db.y >> 24) & 255, (dk.y >> 24) & 255);
    double total = 0.0;
    for (int twoJ = Jlo; twoJ <= Jhi; twoJ += 2) {
        int lb = max(J12minb, abs(twoJ - jc) >> 1), hb = min((db.y >> 8) & 255, (twoJ + jc) >> 1);
        int lk = max(J12mink, abs(twoJ - jf) >> 1), hk = min((dk.y >> 8) & 255, (twoJ + jf) >> 1);
        int nb = hb - lb + 1, nk = hk - lk + 1;
        if (nb <= 0 || nk <= 0) continue;
        const int pitch = row_pitch3(nk);
        if (twoJ < aM) { row += (size_t)nb * pitch; continue; }
        double tj = 0.0;
        for (int J12 = lb; J12 <= hb; J12++) {
            double cb = 0.0;
            if (abs(twoM12b) <= 2 * J12) {
                const double* c2 = T.cg2 + __ldg(T.cg2_off + J12 * nj + (jc >> 1));
                int iJ = (twoJ - abs(2 * J12 - jc)) >> 1;
                cb = __ldg(c1b + (J12 - J12minb) * S1b) *
                     __ldg(c2 + (iJ * (2 * J12 + 1) + ((twoM12b + 2 * J12) >> 1)) * (jc + 1) + B.imc);
            }
            double acc = 0.0;
            for (int J12p = lk; J12p <= hk; J12p++) {
                double ck = 0.0;
                if (abs(twoM12k) <= 2 * J12p) {
                    const double* c2 = T.cg2 + __ldg(T.cg2_off + J12p * nj + (jf >> 1));
                    int iJ = (twoJ - abs(2 * J12p - jf)) >> 1;
                    ck = __ldg(c1k + (J12p - J12mink) * S1k) *
                         __ldg(c2 + (iJ * (2 * J12p + 1) + ((twoM12k + 2 * J12p) >> 1)) * (jf + 1) + K.imc);
                }
                const double* cell = row + (J12p - lk);
                double inner = w0 * __ldg(cell);
                inner = fma(w1, __ldg(cell + plane), inner);
                inner = fma(w2, __ldg(cell + 2 * plane), inner);
                inner = fma(w3, __ldg(cell + 3 * plane), inner);
                inner = fma(w4, __ldg(cell + 4 * plane), inner);
                acc = fma(ck, inner, acc);
            }
            tj = fma(cb, acc, tj);
            row += pitch;
        }
        total += tj;
    }
    return (B.sign * K.sign) * total;
}

// s_desc / s_c1off: the tuple descriptors and the stage-1 block offsets in shared memory, or NULL (a variant of the kernel
// below with these tables, the SPS records and the tuple map in shared memory ran no faster: 2.69 ms either way at 2^26)
__device__ __forceinline__ double eval2_naive(const Tables& T, const Side2& B, const Side2& K, int& mask, const int4* s_desc = nullptr,
                                              const int32_t* s_c1off = nullptr)
{
    mask = 0;
    if (!select2(B, K)) return 0.0;
    const int4 db = s_desc ? s_desc[B.tup] : __ldg(T.tdesc2 + B.tup), dk = s_desc ? s_desc[K.tup] : __ldg(T.tdesc2 + K.tup);
    if (!mask2(B, db, dk)) return 0.0;   // implies a common J, i.e. a slab
    const uint32_t so = __ldg(T.slab_off2 + (size_t)B.tup * T.n_tup2 + K.tup);
    mask = 1;
    const int ja = db.x & 255, jb = (db.x >> 8) & 255, jc = dk.x & 255, jd = (dk.x >> 8) & 255;
    const double w0 = T.iso2[B.tz][0] * T.iso2[K.tz][0], w1 = T.iso2[B.tz][1] * T.iso2[K.tz][1];
    const int nj = T.nj;
    const int Jminb = db.y & 255, Jmink = dk.y & 255;
    const int ob = (ja >> 1) * nj + (jb >> 1), ok = (jc >> 1) * nj + (jd >> 1);
    const double* cb = T.cg1 + (s_c1off ? s_c1off[ob] : __ldg(T.cg1_off + ob)) + B.ima * (jb + 1) + B.imb;
    const double* ck = T.cg1 + (s_c1off ? s_c1off[ok] : __ldg(T.cg1_off + ok)) + K.ima * (jd + 1) + K.imb;
    const int Sb = (ja + 1) * (jb + 1), Sk = (jc + 1) * (jd + 1);
    const int Jlo = max(Jminb, Jmink), Jhi = min((db.y >> 8) & 255, (dk.y >> 8) & 255);
    const double2* cell = (const double2*)(T.slab2 + (size_t)so * CELL2);
    double total = 0.0;
    for (int J = Jlo; J <= Jhi; J++) {
        double2 v = __ldg(cell + (J - Jlo));
        double c = __ldg(cb + (J - Jminb) * Sb) * __ldg(ck + (J - Jmink) * Sk);
        total = fma(c, fma(w1, v.y, w0 * v.x), total);
    }
    double norm = ((db.x >> 24) & 1) ? (((dk.x >> 24) & 1) ? 2.0 : 1.4142135623730951)
                                     : (((dk.x >> 24) & 1) ? 1.4142135623730951 : 1.0);
    return (B.sign * K.sign) * norm * total;
}

template <int BODY>
__global__ void __launch_bounds__(128) k_mscheme_naive(Tables T, long long n, const int32_t* __restrict__ req,
                                                      double* __restrict__ out, uint8_t* __restrict__ maskout, int u16)
{
    long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s[6];
    if (BODY == 3) load_req3(req, i, s, u16); else load_req2(req, i, s, u16);
    double v = 0.0;
    int mask = 0;
    if (!in_range(T, s, 2 * BODY)) {
        atomicAdd(T.bad_count, 1ull);
    } else if (BODY == 3) {
        Side3 B = decode3<false>(T, T.sps_rec, nullptr, s[0], s[1], s[2]), K = decode3<false>(T, T.sps_rec, nullptr, s[3], s[4], s[5]);
        v = eval3_naive(T, B, K, mask);
    } else {
        Side2 B = decode2<false>(T, T.sps_rec, s[0], s[1]), K = decode2<false>(T, T.sps_rec, s[2], s[3]);
        v = eval2_naive(T, B, K, mask);
    }
    out[i] = mask ? v : 0.0;
    if (maskout) maskout[i] = (uint8_t)mask;
}

// 3-body, thread per request on the library's own tables: the coefficient products dtab3 and the isospin-combined slabs vw20
// instead of two CG factors and five planes per term (3 loads per cell instead of 7).  This is what the library takes by
// itself for small 3-body batches (chunks of ~20 000 requests), where the group sort's per-call cost (memset and
// scan of all sort buckets, the pass over all n_tup^2 groups) exceeds the work.  Same operations in the same order as
// small_group3 / k_transform3 (and hence as k_mscheme_naive): bit-identical values.
__global__ void __launch_bounds__(128) k_direct3(Tables T, long long n, const int32_t* __restrict__ req, double* __restrict__ out,
                                                uint8_t* __restrict__ maskout, int u16)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    int s[6];
    load_req3(req, i, s, u16);
    double v = 0.0;
    int mask = 0;
    if (!in_range(T, s, 6)) {
        atomicAdd(T.bad_count, 1ull);
    } else {
        const Side3 B = decode3<false>(T, T.sps_rec, nullptr, s[0], s[1], s[2]), K = decode3<false>(T, T.sps_rec, nullptr, s[3], s[4], s[5]);
        if (select3(T, B, K)) {
            const uint4 sg = __ldg(T.sgrp3 + (size_t)B.tup * T.n_tup3 + K.tup);
            const int4 db = __ldg(T.tdesc3 + B.tup), dk = __ldg(T.tdesc3 + K.tup);
            if (sg.x != NO_SLAB && mask3(T.stmask3, B, K, db, dk)) {
                mask = 1;
                const int4 kb = __ldg(T.tk3 + B.tup), kk = __ldg(T.tk3 + K.tup);
                const int jb1 = ((db.x >> 8) & 255) + 1, jc1 = ((db.x >> 16) & 255) + 1;
                const int je1 = ((dk.x >> 8) & 255) + 1, jf1 = ((dk.x >> 16) & 255) + 1;
                const uint32_t sb = __ldg(T.sig3 + db.w + (B.ima * jb1 + B.imb) * jc1 + B.imc);
                const uint32_t sk = __ldg(T.sig3 + dk.w + (K.ima * je1 + K.imb) * jf1 + K.imc);
                const uint32_t bin = __ldg(T.tz2bin3 + ((B.tz << 3) | K.tz));
                const uint32_t gsize = sg.y;
                const uint32_t* __restrict__ vwb = T.vw20 + (size_t)sg.z * 4 + (size_t)bin * vw_stride(gsize, T.vw_f32);
                const int Jminb = (kb.w >> 16) & 255, Jmink = (kk.w >> 16) & 255;
                const int Jlo = max(Jminb, Jmink), Jhi = min((kb.w >> 24) & 255, (kk.w >> 24) & 255);
                const int2* __restrict__ jib = T.jinfo3 + kb.z + ((Jlo - Jminb) >> 1);
                const int2* __restrict__ jik = T.jinfo3 + kk.z + ((Jlo - Jmink) >> 1);
                const double* __restrict__ dtab = T.dtab3;
                const int aM = abs(B.twoM);
                uint32_t c = 0;   // first Vw cell of the J block
                double total = 0.0;
                for (int twoJ = Jlo, q = 0; twoJ <= Jhi; twoJ += 2, q++) {
                    const int2 ib = __ldg(jib + q), ik = __ldg(jik + q);
                    const int nb = ib.y, nk = ik.y;
                    if (nb <= 0 || nk <= 0) continue;
                    const uint32_t P = (uint32_t)row_pitch3(nk);
                    if (twoJ >= aM) {   // below |M| every coefficient of the block is zero
                        const double* __restrict__ bp = dtab + ((uint32_t)kb.x + (uint32_t)ib.x + sb * (uint32_t)nb);
                        const double* __restrict__ kp = dtab + ((uint32_t)kk.x + (uint32_t)ik.x + sk * (uint32_t)nk);
                        double t = 0.0;
                        for (int r = 0; r < nb; r++) {
                            double acc = 0.0;
                            for (int k = 0; k < nk; k++) {
                                const double ck = __ldg(kp + k), x = ldvw_global(vwb, gsize, c + (uint32_t)r * P + (uint32_t)k, T.vw_f32);
                                acc = k ? fma(ck, x, acc) : ck * x;
                            }
                            t = fma(__ldg(bp + r), acc, t);
                        }
                        total += t;
                    }
                    c += (uint32_t)nb * P;
                }
                v = (B.sign * K.sign < 0 ? -total : total) + 0.0;
            }
        }
    }
    out[i] = mask ? v : 0.0;
    if (maskout) maskout[i] = (uint8_t)mask;
}

// =============================================================================== H1: records
// One thread per request: decode, S1-S7 -> mask (request order, coalesced), canonical packed record.
// Blocks walk KEYS_PER_BLOCK consecutive requests.  With SMEM the small per-basis tables every request needs (SPS
// records, the (a,b) -> tuple map) are copied to shared memory once per block: a random 4..16-byte
// look-up there costs a few bank-conflict wavefronts instead of up to 32 L1 tag look-ups (ncu: k_keys was bound by
// the L1 data pipe, 81 % of peak).
// Sort path: a block also counts its tile's records per COARSE bin (bucket >> csh, at most PART_NC bins) in shared memory
// and leaves the counts in tcnt[tile][bin] for the two-pass partition below (no global atomics for it).
constexpr int KEYS_SPS_SMEM = 2048, KEYS_AB_SMEM = 2048, KEYS_PER_BLOCK = 256 * 32;
constexpr int PART_NC = 2048;
static_assert(KEYS_SPS_SMEM <= 2048 && KEYS_AB_SMEM <= 64 * 64 && 3 * MAX_TWOJ <= 63, "field widths of sps_pack_sorted");
#ifndef MFDN_DIRECT3_MAX
#define MFDN_DIRECT3_MAX (1ll << 20)    // 3-body batches up to this size are evaluated thread-per-request (k_direct3); twice that
                                        // if the isospin-combined slabs are under 64 MB (cache-resident: config 2, 1.44 M requests)
#endif
#ifndef MFDN_TWO_PASS_MIN
#define MFDN_TWO_PASS_MIN (1ll << 23)   // requests from which the two-pass partition beats the one-pass scatter / gather
#endif

template <int BODY, bool AGG, bool SMEM>
__global__ void __launch_bounds__(256) k_keys(Tables T, long long n, const int32_t* __restrict__ req,
                                              unsigned long long* __restrict__ recs, uint8_t* __restrict__ maskout,
                                              uint32_t* __restrict__ hist, uint32_t invalid_bucket,
                                              uint32_t* __restrict__ keys32, uint32_t* __restrict__ tcnt, int csh, int nc, int u16)
{
    __shared__ uint32_t s_sps[SMEM ? KEYS_SPS_SMEM : 1];
    __shared__ int2 s_ab[SMEM && BODY == 3 ? KEYS_AB_SMEM : 1];
    __shared__ uint32_t s_ch[AGG ? 1 : PART_NC];
    if (!AGG && tcnt) {
        for (int k = threadIdx.x; k < nc; k += blockDim.x) s_ch[k] = 0u;
        if (!SMEM) __syncthreads();
    }
    if (SMEM) {
        for (int k = threadIdx.x; k < T.n_sps; k += blockDim.x) s_sps[k] = __ldg(T.sps_rec + k);
        if (BODY == 3) {
            for (int k = threadIdx.x; k < T.n_orb * T.n_orb; k += blockDim.x) s_ab[k] = __ldg(T.ab3 + k);
        }
        __syncthreads();
    }
    const uint32_t* sps = SMEM ? s_sps : T.sps_rec;
    const int2* ab = (SMEM && BODY == 3) ? s_ab : nullptr;
    const long long i0 = (long long)blockIdx.x * KEYS_PER_BLOCK + threadIdx.x;
    const long long i1 = min(n, (long long)(blockIdx.x + 1) * KEYS_PER_BLOCK);
    int nx[6];
    if (i0 < i1) { if (BODY == 3) load_req3(req, i0, nx, u16); else load_req2(req, i0, nx, u16); }
    for (long long i = i0; i < i1; i += 256) {
        int s[6];
#pragma unroll
        for (int k = 0; k < 6; k++) s[k] = nx[k];
        if (i + 256 < i1) { if (BODY == 3) load_req3(req, i + 256, nx, u16); else load_req2(req, i + 256, nx, u16); }   // next request in flight
        uint32_t key = REC_INVALID;
        unsigned long long low = 0;
        int mask = 0;
        if (!in_range(T, s, 2 * BODY)) {
            if (recs) atomicAdd(T.bad_count, 1ull);
        } else if (BODY == 3) {
            Side3 B = decode3<SMEM>(T, sps, ab, s[0], s[1], s[2]), K = decode3<SMEM>(T, sps, ab, s[3], s[4], s[5]);
            if (select3(T, B, K)) {
                const int4 db = __ldg(T.tdesc3 + B.tup), dk = __ldg(T.tdesc3 + K.tup);
                {   // sort key = (group, M) bucket: the group's first bucket + index of M in the common M range
                    const int sjb = (db.x & 255) + ((db.x >> 8) & 255) + ((db.x >> 16) & 255);
                    const int sjk = (dk.x & 255) + ((dk.x >> 8) & 255) + ((dk.x >> 16) & 255);
                    key = __ldg(T.gbase3 + (size_t)B.tup * T.n_tup3 + K.tup) + (uint32_t)(B.ima + B.imb + B.imc - ((sjb - min(sjb, sjk)) >> 1));
                }
                mask = mask3(T.stmask3, B, K, db, dk);
                const int jb1 = ((db.x >> 8) & 255) + 1, jc1 = ((db.x >> 16) & 255) + 1;
                const int je1 = ((dk.x >> 8) & 255) + 1, jf1 = ((dk.x >> 16) & 255) + 1;
                const uint32_t sb = __ldg(T.sig3 + db.w + (B.ima * jb1 + B.imb) * jc1 + B.imc);
                const uint32_t sk = __ldg(T.sig3 + dk.w + (K.ima * je1 + K.imb) * jf1 + K.imc);
                const uint32_t bin = __ldg(T.tz2bin3 + ((B.tz << 3) | K.tz));
                low = (unsigned long long)(sb | (sk << 12) | (bin << 24) | ((uint32_t)(B.sign * K.sign < 0) << 29)) |
                      ((unsigned long long)(B.ima + B.imb + B.imc) << 30);
            }
        } else {
            Side2 B = decode2<SMEM>(T, sps, s[0], s[1]), K = decode2<SMEM>(T, sps, s[2], s[3]);
            if (select2(B, K)) {
                key = (uint32_t)B.tup * T.n_tup2 + K.tup;
                // a group without a slab (no common J) has no common channel either: mask2 alone decides, no n_tup^2 gather
                mask = mask2(B, __ldg(T.tdesc2 + B.tup), __ldg(T.tdesc2 + K.tup));
                low = (unsigned long long)(B.ima | (B.imb << 5) | (K.ima << 15) | (K.imb << 20)) |
                      ((unsigned long long)((B.tz << 3) | K.tz) << 30) | ((unsigned long long)(B.sign * K.sign < 0) << 36);
            }
        }
        if (recs) recs[i] = ((unsigned long long)key << REC_KEY_SHIFT) | low;
        if (maskout) maskout[i] = (uint8_t)mask;
        if (hist) {
            const uint32_t bucket = key == REC_INVALID ? invalid_bucket : key;
            if (AGG) {   // group-ordered input: one atomic per run of equal keys in the warp
                const unsigned act = __activemask();
                const unsigned same = __match_any_sync(act, bucket);
                if ((threadIdx.x & 31) == __ffs(same) - 1) atomicAdd(hist + bucket, (uint32_t)__popc(same));
            } else {
                atomicAdd(hist + bucket, 1u);
                if (tcnt) atomicAdd(&s_ch[bucket >> csh], 1u);
            }
        }
        if (keys32) keys32[i] = key == REC_INVALID ? 0xFFFFFFFFu : key;
    }
    if (!AGG && tcnt) {
        __syncthreads();
        for (int k = threadIdx.x; k < nc; k += blockDim.x) tcnt[(size_t)blockIdx.x * nc + k] = s_ch[k];
    }
}

// H1, 3-body, every per-basis table in shared memory: SPS records, (a,b) -> tuple map, tuple descriptors, the two small
// tables that give a group's first sort bucket (rowbase3 + colcum3 instead of a gather from the n_tup^2 array gbase3), the
// per-class sigma maps and the tz -> isospin-bin map.  ncu on k_keys: L1 data pipe 89 % busy, a gather of 32 random table
// entries costs up to 32 L1 wavefronts against 3-4 bank-conflict wavefronts in shared memory; without the sigma and the
// bucket gathers the kernel ran in 1.10 instead of 1.39 ms each (n = 2^26).  One persistent block per SM walks the tiles
// (the tables are loaded once).  The S7 state masks, deduplicated at upload, are there too (0.21 ms of gathers otherwise).
constexpr int KS_THREADS = 1024;
struct KeysSmem3 {   // byte offsets into the dynamic shared memory, filled by the host
    uint32_t tdesc, stm, ab, sps, rowbase, ch, colcum, sig, tzbin, total;
};
template <bool AGG, bool U16>
__global__ void __launch_bounds__(KS_THREADS, 1) k_keys3s(Tables T, KeysSmem3 L, long long n, const int32_t* __restrict__ req,
                                                         unsigned long long* __restrict__ recs, uint8_t* __restrict__ maskout,
                                                         uint32_t* __restrict__ hist, uint32_t invalid_bucket,
                                                         uint32_t* __restrict__ tcnt, int csh, int nc, int n_tiles)
{
    extern __shared__ __align__(16) unsigned char ks_smem[];
    int4* s_tdesc = reinterpret_cast<int4*>(ks_smem + L.tdesc);
    unsigned long long* s_stm = reinterpret_cast<unsigned long long*>(ks_smem + L.stm);
    int2* s_ab = reinterpret_cast<int2*>(ks_smem + L.ab);
    uint32_t* s_sps = reinterpret_cast<uint32_t*>(ks_smem + L.sps);
    uint32_t* s_rowbase = reinterpret_cast<uint32_t*>(ks_smem + L.rowbase);
    uint32_t* s_ch = reinterpret_cast<uint32_t*>(ks_smem + L.ch);
    uint16_t* s_colcum = reinterpret_cast<uint16_t*>(ks_smem + L.colcum);
    uint16_t* s_sig = reinterpret_cast<uint16_t*>(ks_smem + L.sig);
    uint8_t* s_tzbin = ks_smem + L.tzbin;
    const int tid = threadIdx.x, nt = T.n_tup3;
    for (int k = tid; k < nt; k += KS_THREADS) {
        int4 d = __ldg(T.tdesc3 + k);
        d.z = __ldg(T.stm12_off3 + k);   // this kernel's copy: offset in the direct S7 table instead of in stmask3
        s_tdesc[k] = d;
        s_rowbase[k] = __ldg(T.rowbase3 + k);
    }
    for (int k = tid; k < T.stm12_len3; k += KS_THREADS) s_stm[k] = __ldg(T.stm12_3 + k);
    for (int k = tid; k < T.n_orb * T.n_orb; k += KS_THREADS) s_ab[k] = __ldg(T.ab3 + k);
    for (int k = tid; k < T.n_sps; k += KS_THREADS) s_sps[k] = sps_pack_sorted(__ldg(T.sps_rec + k), k);
    for (int k = tid; k < T.ncls3 * nt; k += KS_THREADS) s_colcum[k] = __ldg(T.colcum3 + k);
    for (int k = tid; k < T.sig_len3; k += KS_THREADS) s_sig[k] = __ldg(T.sig3 + k);
    if (tid < 64) s_tzbin[tid] = __ldg(T.tz2bin3 + tid);
    // the coarse counts are double-buffered: ONE block barrier per tile (the counts of tile t are flushed and zeroed while tile
    // t + 1 is counted into the other half; the barrier was 14 % of the stall samples on the skewed config-4 stream)
    if (tcnt)
        for (int k = tid; k < 2 * nc; k += KS_THREADS) s_ch[k] = 0u;
    __syncthreads();   // also: the tables are loaded
    uint32_t* s_cur = s_ch;
    for (int tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long i0 = (long long)tile * KEYS_PER_BLOCK + tid;
        const long long i1 = min(n, (long long)(tile + 1) * KEYS_PER_BLOCK);
        int nx[6];
        if (i0 < i1) load_req3(req, i0, nx, U16);
        for (long long i = i0; i < i1; i += KS_THREADS) {
            int s[6];
#pragma unroll
            for (int k = 0; k < 6; k++) s[k] = nx[k];
            if (i + KS_THREADS < i1) load_req3(req, i + KS_THREADS, nx, U16);   // next request in flight
            uint32_t key = REC_INVALID;
            unsigned long long low = 0;
            int mask = 0;
            if (max(max((unsigned)s[0], (unsigned)s[1]), max(max((unsigned)s[2], (unsigned)s[3]), max((unsigned)s[4], (unsigned)s[5]))) >= (unsigned)T.n_sps) {
                atomicAdd(T.bad_count, 1ull);
            } else {
                Side3 B = decode3s(T, s_sps, s_ab, s[0], s[1], s[2]), K = decode3s(T, s_sps, s_ab, s[3], s[4], s[5]);
                if (select3(T, B, K)) {
                    const int4 db = s_tdesc[B.tup], dk = s_tdesc[K.tup];
                    const int sjb = (db.x & 255) + ((db.x >> 8) & 255) + ((db.x >> 16) & 255);
                    const int sjk = (dk.x & 255) + ((dk.x >> 8) & 255) + ((dk.x >> 16) & 255);
                    key = s_rowbase[B.tup] + s_colcum[((db.x >> 26) & 31) * nt + K.tup] +
                          (uint32_t)(B.ima + B.imb + B.imc - ((sjb - min(sjb, sjk)) >> 1));
                    mask = mask3s(s_stm, B, K, db.z, dk.z);
                    const int jb1 = ((db.x >> 8) & 255) + 1, jc1 = ((db.x >> 16) & 255) + 1;
                    const int je1 = ((dk.x >> 8) & 255) + 1, jf1 = ((dk.x >> 16) & 255) + 1;
                    const uint32_t sb = s_sig[db.w + (B.ima * jb1 + B.imb) * jc1 + B.imc];
                    const uint32_t sk = s_sig[dk.w + (K.ima * je1 + K.imb) * jf1 + K.imc];
                    const uint32_t bin = s_tzbin[(B.tz << 3) | K.tz];
                    low = (unsigned long long)(sb | (sk << 12) | (bin << 24) | ((uint32_t)(B.sign * K.sign < 0) << 29)) |
                          ((unsigned long long)(B.ima + B.imb + B.imc) << 30);
                }
            }
            recs[i] = ((unsigned long long)key << REC_KEY_SHIFT) | low;
            if (maskout) maskout[i] = (uint8_t)mask;
            const uint32_t bucket = key == REC_INVALID ? invalid_bucket : key;
            if (AGG) {   // group-ordered input: one atomic per run of equal keys in the warp (runs found with shfl.up + ballot
                         // instead of match.any: pre-sorted call 2.005 -> 2.05 ms, not kept)
                const unsigned same = __match_any_sync(__activemask(), bucket);
                if ((tid & 31) == __ffs(same) - 1) atomicAdd(hist + bucket, (uint32_t)__popc(same));
            } else {
                if (hist) atomicAdd(hist + bucket, 1u);   // NULL: the buckets are counted per pass-2 tile (k_count2) instead
                if (tcnt) atomicAdd(&s_cur[bucket >> csh], 1u);
            }
        }
        if (tcnt) {
            __syncthreads();
            for (int k = tid; k < nc; k += KS_THREADS) {
                tcnt[(size_t)tile * nc + k] = s_cur[k];
                s_cur[k] = 0u;   // used again two tiles from now, after the next barrier
            }
            s_cur = s_cur == s_ch ? s_ch + nc : s_ch;
        }
    }
}

// =============================================================================== H2: group sort
// exclusive scan of v over the threads of a block of NT threads (NT a multiple of 32, at most 1024); `total` = sum
template <int NT>
__device__ __forceinline__ uint32_t block_excl_scan(uint32_t v, uint32_t* s_warp /* [NT / 32 + 1] */, uint32_t& total)
{
    const int tid = threadIdx.x;
    uint32_t inc = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, inc, off);
        if ((tid & 31) >= off) inc += x;
    }
    __syncthreads();   // s_warp may still be read from a previous call
    if ((tid & 31) == 31) s_warp[tid >> 5] = inc;
    __syncthreads();
    if (tid < 32) {
        const uint32_t w = tid < NT / 32 ? s_warp[tid] : 0u;
        uint32_t wi = w;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, wi, off);
            if (tid >= off) wi += x;
        }
        if (tid < NT / 32) s_warp[tid] = wi - w;
        if (tid == 31) s_warp[NT / 32] = wi;
    }
    __syncthreads();
    total = s_warp[NT / 32];
    return s_warp[tid >> 5] + inc - v;
}

constexpr int SCAN_T = 256, SCAN_E = 16, SCAN_TILE = SCAN_T * SCAN_E;

__global__ void __launch_bounds__(SCAN_T) k_scan_tiles(uint32_t* __restrict__ data, long long m, uint32_t* __restrict__ tile_sums)
{
    __shared__ uint32_t s_warp[SCAN_T / 32 + 1];
    long long base = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_E;
    uint32_t v[SCAN_E], sum = 0;
    const bool full = base + SCAN_E <= m;   // the thread's 16 words as four 128-bit accesses (data is 256-byte aligned)
    if (full) {
#pragma unroll
        for (int k = 0; k < SCAN_E / 4; k++) {
            const uint4 q = reinterpret_cast<const uint4*>(data + base)[k];
            v[4 * k] = q.x; v[4 * k + 1] = q.y; v[4 * k + 2] = q.z; v[4 * k + 3] = q.w;
        }
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_E; k++) v[k] = (base + k < m) ? data[base + k] : 0u;
    }
#pragma unroll
    for (int k = 0; k < SCAN_E; k++) sum += v[k];
    uint32_t all;
    uint32_t excl = block_excl_scan<SCAN_T>(sum, s_warp, all);   // warp shuffles, three block barriers
    if (threadIdx.x == 0) tile_sums[blockIdx.x] = all;
    if (full) {
#pragma unroll
        for (int k = 0; k < SCAN_E / 4; k++) {
            uint4 q;
            q.x = excl; excl += v[4 * k];
            q.y = excl; excl += v[4 * k + 1];
            q.z = excl; excl += v[4 * k + 2];
            q.w = excl; excl += v[4 * k + 3];
            reinterpret_cast<uint4*>(data + base)[k] = q;
        }
    } else {
#pragma unroll
        for (int k = 0; k < SCAN_E; k++) {
            if (base + k < m) data[base + k] = excl;
            excl += v[k];
        }
    }
}

__global__ void __launch_bounds__(1024) k_scan_sums(uint32_t* __restrict__ sums, int n_tiles)
{
    __shared__ uint32_t sh[1024];
    uint32_t carry = 0;
    for (int base = 0; base < n_tiles; base += 1024) {
        int i = base + threadIdx.x;
        uint32_t v = i < n_tiles ? sums[i] : 0u;
        sh[threadIdx.x] = v;
        __syncthreads();
        for (int off = 1; off < 1024; off <<= 1) {
            uint32_t x = threadIdx.x >= off ? sh[threadIdx.x - off] : 0u;
            __syncthreads();
            sh[threadIdx.x] += x;
            __syncthreads();
        }
        if (i < n_tiles) sums[i] = carry + sh[threadIdx.x] - v;
        carry += sh[1023];
        __syncthreads();
    }
}

__global__ void __launch_bounds__(SCAN_T) k_scan_add(uint32_t* __restrict__ data, long long m, const uint32_t* __restrict__ tile_sums)
{
    uint32_t add = tile_sums[blockIdx.x];
    long long base = (long long)blockIdx.x * SCAN_TILE + (long long)threadIdx.x * SCAN_E;
    if (base + SCAN_E <= m) {
#pragma unroll
        for (int k = 0; k < SCAN_E / 4; k++) {
            uint4 q = reinterpret_cast<uint4*>(data + base)[k];
            q.x += add; q.y += add; q.z += add; q.w += add;
            reinterpret_cast<uint4*>(data + base)[k] = q;
        }
        return;
    }
#pragma unroll
    for (int k = 0; k < SCAN_E; k++)
        if (base + k < m) data[base + k] += add;
}

// H2 group sort and H6 gather back = a two-pass partition of the 8-byte records and its mirror image for the values.
// What decides the speed of a permutation of 2^26 8-byte elements on this machine is the number of sectors a memory
// instruction touches, not DRAM locality: a store (or load) whose 32 lanes hit 32 different sectors costs 32 L1
// wavefronts and 32 L2 requests, and the one-pass forms ran at 50-75 G elements/s whatever the window they wrote into
// (measured at n = 2^26: one-pass scatter 1.71 ms, gather 1.06 ms; a two-pass partition with direct 8-byte stores 1.06 +
// 1.38 ms; the same first pass staged in shared memory 0.33 ms).  So every pass below permutes a TILE in shared memory
// first and then moves runs of consecutive elements with consecutive lanes:
//   pass 1 (k_part1)  tile of KEYS_PER_BLOCK requests -> coarse bins (bucket >> csh).  The tile's first position in
//           every bin comes from tcnt (k_keys' per-tile counts, exclusive-scanned over the tiles by k_tscan_*): no
//           global atomics, the (tile, bin) runs are contiguous.  Leaves map1[tile slot] = coarse-order position and
//           slot1[request] = tile slot for the way back.
//   pass 2 (k_part2)  tiles of the coarse-ordered stream that do not straddle a coarse bin (k_tiles2) -> buckets: local
//           counting in shared memory, one global atomic per (tile, non-empty bucket) on the scanned histogram, runs
//           written to their final place.  Leaves map2 / slot2 likewise.  The cursor array ends up holding bucket ENDS.
//   transform          reads the bucket-ordered records, writes the values in the same order (coalesced).
//   H6a (k_back<2>)    per pass-2 tile: values of its runs -> shared memory -> coarse order.
//   H6b (k_back<1>)    per pass-1 tile: values of its runs -> shared memory -> request order.
// Capacity: PART_NC coarse bins x PART_NF buckets per bin; tables with more (group, M) buckets than that take the
// one-pass scatter / gather (k_scatter, k_unpermute) instead.
constexpr int SC_PER_THREAD = 4;
constexpr int TS_CHUNK = 64;      // tiles per chunk of the two-level scan over the tiles
constexpr int PART_NF = 4096;     // buckets per coarse bin, at most
#ifndef MFDN_P_THREADS
#define MFDN_P_THREADS 512
#endif
constexpr int P_THREADS = MFDN_P_THREADS;
constexpr int PART_SMEM = KEYS_PER_BLOCK * 8 + 2 * PART_NF * 4;   // staged tile + two tables of max(PART_NC, PART_NF) words
static_assert(PART_NC <= PART_NF && KEYS_PER_BLOCK <= 65536, "table sizes / 16-bit tile slots");

// part[chunk][bin] = sum of tcnt over the chunk's tiles
__global__ void __launch_bounds__(128) k_tscan_sum(const uint32_t* __restrict__ tcnt, int n_tiles, int nc, uint32_t* __restrict__ part)
{
    const int c = blockIdx.x * 128 + threadIdx.x, k = blockIdx.y;
    if (c >= nc) return;
    const int t0 = k * TS_CHUNK, t1 = min(n_tiles, t0 + TS_CHUNK);
    uint32_t sum = 0;
#pragma unroll 16
    for (int t = t0; t < t1; t++) sum += __ldg(tcnt + (size_t)t * nc + c);
    part[(size_t)k * nc + c] = sum;
}


// part[chunk][bin] -> records of the bin in the chunks before (exclusive scan over chunks); cstart[bin] = start of the bin
// in the coarse-ordered stream, cstart[nc] = n
__global__ void __launch_bounds__(1024) k_tscan_mid(uint32_t* __restrict__ part, int n_chunks, int nc, uint32_t* __restrict__ cstart)
{
    __shared__ uint32_t s_warp[33];
    uint32_t carry = 0;
    for (int c0 = 0; c0 < nc; c0 += 1024) {
        const int c = c0 + threadIdx.x;
        uint32_t total = 0;
        if (c < nc) {
            for (int k0 = 0; k0 < n_chunks; k0 += 16) {
                uint32_t v[16];
#pragma unroll
                for (int u = 0; u < 16; u++) v[u] = k0 + u < n_chunks ? part[(size_t)(k0 + u) * nc + c] : 0u;
#pragma unroll
                for (int u = 0; u < 16; u++) {
                    if (k0 + u < n_chunks) part[(size_t)(k0 + u) * nc + c] = total;
                    total += v[u];
                }
            }
        }
        uint32_t all;
        const uint32_t start = carry + block_excl_scan<1024>(total, s_warp, all);
        carry += all;
        if (c < nc) cstart[c] = start;
    }
    if (threadIdx.x == 0) cstart[nc] = carry;
}
// tcnt[tile][bin] -> first position of the tile in the bin
__global__ void __launch_bounds__(128) k_tscan_fill(uint32_t* __restrict__ tcnt, int n_tiles, int nc, const uint32_t* __restrict__ part,
                                                    const uint32_t* __restrict__ cstart)
{
    const int c = blockIdx.x * 128 + threadIdx.x, k = blockIdx.y;
    if (c >= nc) return;
    const int t0 = k * TS_CHUNK, t1 = min(n_tiles, t0 + TS_CHUNK);
    uint32_t run = part[(size_t)k * nc + c] + cstart[c];
    for (int ta = t0; ta < t1; ta += 16) {
        uint32_t v[16];
#pragma unroll
        for (int u = 0; u < 16; u++) v[u] = ta + u < t1 ? tcnt[(size_t)(ta + u) * nc + c] : 0u;
#pragma unroll
        for (int u = 0; u < 16; u++) {
            if (ta + u < t1) tcnt[(size_t)(ta + u) * nc + c] = run;
            run += v[u];
        }
    }
}
// pass-2 tiles: every coarse bin is cut into tiles of at most KEYS_PER_BLOCK records: tiles2[1 + k] = {first position,
// records, bin, 0}; tiles2[0].x = number of tiles
__global__ void __launch_bounds__(1024) k_tiles2(const uint32_t* __restrict__ cstart, int nc, uint4* __restrict__ tiles2)
{
    __shared__ uint32_t s_warp[33];
    uint32_t carry = 0;
    for (int c0 = 0; c0 < nc; c0 += 1024) {
        const int c = c0 + threadIdx.x;
        uint32_t s = 0, e = 0;
        if (c < nc) { s = cstart[c]; e = cstart[c + 1]; }
        const uint32_t k = (e - s + KEYS_PER_BLOCK - 1) / KEYS_PER_BLOCK;
        uint32_t all;
        const uint32_t first = carry + block_excl_scan<1024>(k, s_warp, all);
        carry += all;
        for (uint32_t j = 0; j < k; j++)
            tiles2[1 + first + j] = make_uint4(s + j * KEYS_PER_BLOCK, min((uint32_t)KEYS_PER_BLOCK, e - s - j * KEYS_PER_BLOCK), (uint32_t)c, 0u);
    }
    if (threadIdx.x == 0) tiles2[0] = make_uint4(carry, 0u, 0u, 0u);
}

__device__ __forceinline__ uint32_t rec_bucket(unsigned long long r, uint32_t invalid_bucket)
{
    const uint32_t key = (uint32_t)(r >> REC_KEY_SHIFT);
    return key == REC_INVALID ? invalid_bucket : key;
}

// Histogram of the sort buckets from the coarse-ordered stream, one block per pass-2 tile: counted in shared memory, then ONE
// global atomic per (tile, non-empty bucket).  Replaces the per-request histogram atomic of H1 on the two-pass path: on a
// skewed stream those atomics pile up on a few L2 lines (config 4: H1 0.57 ms per 2^24 requests against 0.26 ms on a uniform
// stream over the same tables); here a hot bucket costs one atomic per tile.  Price: the records are read once more.
__global__ void __launch_bounds__(P_THREADS) k_count2(const unsigned long long* __restrict__ p1rec, const uint4* __restrict__ tiles2,
                                                     uint32_t* __restrict__ hist, int csh, uint32_t invalid_bucket)
{
    __shared__ uint32_t s_cnt[PART_NF];
    if (blockIdx.x >= __ldg(&tiles2[0].x)) return;
    const uint4 t = __ldg(tiles2 + 1 + blockIdx.x);
    const uint32_t d0 = t.z << csh;
    const int nd = min(1 << csh, (int)(invalid_bucket + 1u - d0)), m = (int)t.y, tid = threadIdx.x;
    for (int k = tid; k < nd; k += P_THREADS) s_cnt[k] = 0u;
    __syncthreads();
    for (int l = tid; l < m; l += P_THREADS) atomicAdd(&s_cnt[rec_bucket(__ldg(p1rec + t.x + l), invalid_bucket) - d0], 1u);
    __syncthreads();
    for (int k = tid; k < nd; k += P_THREADS) {
        const uint32_t v = s_cnt[k];
        if (v) atomicAdd(hist + d0 + k, v);
    }
}

// One partition pass over one tile.  PASS 1: tile = k_keys tile blockIdx.x, digit = bucket >> csh, first positions from
// toff[tile][digit].  PASS 2: tile = tiles2[1 + blockIdx.x] (inside coarse bin c), digit = bucket - (c << csh), first
// positions reserved on cursor[bucket].  map[tile start + slot] = destination of the tile's slot-th record in digit order,
// slot_of[source position] = slot.
template <int PASS>
__global__ void __launch_bounds__(P_THREADS) k_part(long long n, const unsigned long long* __restrict__ src, const uint32_t* __restrict__ toff,
                                                   const uint4* __restrict__ tiles2, uint32_t* __restrict__ cursor, int csh, int nd,
                                                   unsigned long long* __restrict__ dst, uint32_t* __restrict__ map, uint16_t* __restrict__ slot_of,
                                                   uint32_t invalid_bucket)
{
    extern __shared__ __align__(16) unsigned char part_smem[];
    unsigned long long* stage = reinterpret_cast<unsigned long long*>(part_smem);   // [KEYS_PER_BLOCK]
    uint32_t* s_cnt = reinterpret_cast<uint32_t*>(stage + KEYS_PER_BLOCK);           // [nd] counts, then first slot of the digit
    uint32_t* s_g = s_cnt + PART_NF;                                                 // [nd] destination - slot
    __shared__ uint32_t s_warp[P_THREADS / 32 + 1];
    constexpr int PER = KEYS_PER_BLOCK / P_THREADS;
    const int tid = threadIdx.x;
    long long i0;
    int m;
    uint32_t d0;   // digit = (bucket >> dsh) - d0
    int dsh;
    if (PASS == 1) {
        i0 = (long long)blockIdx.x * KEYS_PER_BLOCK;
        m = (int)min((long long)KEYS_PER_BLOCK, n - i0);
        d0 = 0u; dsh = csh;
    } else {
        if (blockIdx.x >= __ldg(&tiles2[0].x)) return;
        const uint4 t = __ldg(tiles2 + 1 + blockIdx.x);
        i0 = t.x; m = (int)t.y;
        d0 = t.z << csh; dsh = 0;
        nd = min(nd, (int)(invalid_bucket + 1u - d0));   // the last coarse bin may be short
    }
    for (int k = tid; k < nd; k += P_THREADS) s_cnt[k] = 0u;
    __syncthreads();
    unsigned long long r[PER];
    uint32_t rank[PER];
#pragma unroll
    for (int u = 0; u < PER; u++) r[u] = tid + u * P_THREADS < m ? __ldcs(src + i0 + tid + u * P_THREADS) : 0ull;
#pragma unroll
    for (int u = 0; u < PER; u++)
        rank[u] = tid + u * P_THREADS < m ? atomicAdd(&s_cnt[(rec_bucket(r[u], invalid_bucket) >> dsh) - d0], 1u) : 0u;
    __syncthreads();
    // exclusive scan of the counts: thread t owns the digits [t * per, (t + 1) * per)
    {
        const int per = (nd + P_THREADS - 1) / P_THREADS, a = tid * per, b = min(nd, a + per);
        uint32_t sum = 0;
        for (int k = a; k < b; k++) sum += s_cnt[k];
        uint32_t all;
        uint32_t run = block_excl_scan<P_THREADS>(sum, s_warp, all);
        for (int k = a; k < b; k++) {
            const uint32_t v = s_cnt[k];
            s_cnt[k] = run;
            uint32_t g = 0u;
            if (PASS == 1) g = __ldg(toff + (size_t)blockIdx.x * nd + k);
            else if (v) g = atomicAdd(cursor + d0 + k, v);
            s_g[k] = g - run;
            run += v;
        }
    }
    __syncthreads();
#pragma unroll
    for (int u = 0; u < PER; u++) {
        const int l = tid + u * P_THREADS;
        if (l < m) {
            const uint32_t slot = s_cnt[(rec_bucket(r[u], invalid_bucket) >> dsh) - d0] + rank[u];
            stage[slot] = r[u];
            slot_of[i0 + l] = (uint16_t)slot;
        }
    }
    __syncthreads();
    for (int j = tid; j < m; j += P_THREADS) {
        const unsigned long long rc = stage[j];
        const uint32_t to = s_g[(rec_bucket(rc, invalid_bucket) >> dsh) - d0] + (uint32_t)j;
        dst[to] = rc;
        __stcs(map + i0 + j, to);
    }
}

// NEXT-1 epilogue: instead of being returned, result i is multiplied by its stored phase and added to
// the many-body element it pertains to, H[loc[i]] += phase[i] * v[i].  MFDn asks for the 3-body elements of one many-body
// element one after the other, so neighbouring requests often share loc: the lanes of a warp first sum runs of equal
// loc among themselves (segmented scan with shuffles), then the last lane of every run issues ONE fp64 atomic.  Entries
// with loc outside [0, h_len) and exact zeros (mask = 0) are skipped.  All 32 lanes must call this.
struct Accum {
    const long long* loc;
    const double* phase;   // NULL: +1
    double* H;
    long long h_len;
};
__device__ __forceinline__ void accumulate_warp(const Accum& A, long long i, bool valid, double v)
{
    const int lane = threadIdx.x & 31;
    long long l = -1 - lane;   // distinct negative values: lanes without a target never form a run
    double x = 0.0;
    if (valid) {
        const long long t = __ldcs(A.loc + i);
        if (t >= 0 && t < A.h_len) {
            l = t;
            x = A.phase ? __ldcs(A.phase + i) * v : v;
        }
    }
    const long long up = __shfl_up_sync(0xFFFFFFFFu, l, 1);
    const unsigned heads = __ballot_sync(0xFFFFFFFFu, lane == 0 || up != l);
    const int start = 31 - __clz((int)(heads & (0xFFFFFFFFu >> (31 - lane))));   // first lane of this lane's run
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const double y = __shfl_up_sync(0xFFFFFFFFu, x, off);
        if (lane - off >= start) x += y;
    }
    const bool tail = lane == 31 || ((heads >> (lane + 1)) & 1u);
    if (tail && l >= 0 && x != 0.0) atomicAdd(A.H + l, x);
}

// the same for values already in request order (every path but the default one)
__global__ void __launch_bounds__(256) k_accumulate(long long n, const double* __restrict__ vals, Accum A)
{
    const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
    const bool valid = i < n;
    accumulate_warp(A, i, valid, valid ? __ldcs(vals + i) : 0.0);
}

// The way back, one tile of pass PASS per block: vals[map[tile start + slot]] -> shared memory -> out[tile start + l] =
// staged[slot_of[tile start + l]].
// ACC (pass 1 only): the request-order values are not stored but accumulated (NEXT-1), out is unused.
template <int PASS, bool ACC = false>
__global__ void __launch_bounds__(P_THREADS) k_back(long long n, const double* __restrict__ vals, const uint4* __restrict__ tiles2,
                                                   const uint32_t* __restrict__ map, const uint16_t* __restrict__ slot_of, double* __restrict__ out,
                                                   Accum A)
{
    extern __shared__ __align__(16) unsigned char part_smem[];
    double* stage = reinterpret_cast<double*>(part_smem);
    const int tid = threadIdx.x;
    long long i0;
    int m;
    if (PASS == 1) {
        i0 = (long long)blockIdx.x * KEYS_PER_BLOCK;
        m = (int)min((long long)KEYS_PER_BLOCK, n - i0);
    } else {
        if (blockIdx.x >= __ldg(&tiles2[0].x)) return;
        const uint4 t = __ldg(tiles2 + 1 + blockIdx.x);
        i0 = t.x; m = (int)t.y;
    }
    constexpr int PER = KEYS_PER_BLOCK / P_THREADS;
    uint32_t from[PER];
#pragma unroll
    for (int u = 0; u < PER; u++) from[u] = tid + u * P_THREADS < m ? __ldcs(map + i0 + tid + u * P_THREADS) : 0u;
#pragma unroll
    for (int u = 0; u < PER; u++)
        if (tid + u * P_THREADS < m) stage[tid + u * P_THREADS] = __ldcs(vals + from[u]);
    __syncthreads();
    if constexpr (ACC) {
        for (int l0 = 0; l0 < m; l0 += P_THREADS) {   // warp-uniform trip count: every lane takes part in the shuffles
            const int l = l0 + tid;
            const bool valid = l < m;
            accumulate_warp(A, i0 + l, valid, valid ? stage[__ldcs(slot_of + i0 + l)] : 0.0);
        }
    } else {
        for (int l = tid; l < m; l += P_THREADS) {
            const double v = stage[__ldcs(slot_of + i0 + l)];
            if (PASS == 1) __stcs(out + i0 + l, v); else out[i0 + l] = v;
        }
    }
}

// One-pass forms (tables with more buckets than PART_NC x PART_NF): records -> bucket order with one returning atomic
// and one scattered store per request, posof[i] = position of request i; the cursor array ends up holding bucket ENDS.
__global__ void __launch_bounds__(256) k_scatter(long long n, const unsigned long long* __restrict__ recs,
                                                 uint32_t* __restrict__ cursor, unsigned long long* __restrict__ sorted,
                                                 uint32_t* __restrict__ posof, uint32_t invalid_bucket)
{
    const long long base = (long long)blockIdx.x * (256 * SC_PER_THREAD) + threadIdx.x;
    unsigned long long r[SC_PER_THREAD];
    uint32_t pos[SC_PER_THREAD];
#pragma unroll
    for (int u = 0; u < SC_PER_THREAD; u++) {
        const long long i = base + u * 256;
        r[u] = i < n ? __ldcs(recs + i) : 0ull;
    }
#pragma unroll
    for (int u = 0; u < SC_PER_THREAD; u++) {   // SC_PER_THREAD independent atomics in flight per thread
        const long long i = base + u * 256;
        pos[u] = i < n ? atomicAdd(cursor + rec_bucket(r[u], invalid_bucket), 1u) : 0u;
    }
#pragma unroll
    for (int u = 0; u < SC_PER_THREAD; u++) {
        const long long i = base + u * 256;
        if (i < n) {
            sorted[pos[u]] = r[u];
            __stcs(posof + i, pos[u]);
        }
    }
}

// H6, one-pass form: results from bucket order back to request order
__global__ void __launch_bounds__(256) k_unpermute(long long n, const double* __restrict__ vals, const uint32_t* __restrict__ posof,
                                                   double* __restrict__ out)
{
    const long long base = (long long)blockIdx.x * (256 * SC_PER_THREAD) + threadIdx.x;
    uint32_t p[SC_PER_THREAD];
#pragma unroll
    for (int u = 0; u < SC_PER_THREAD; u++) {
        const long long i = base + u * 256;
        p[u] = i < n ? __ldcs(posof + i) : 0u;
    }
#pragma unroll
    for (int u = 0; u < SC_PER_THREAD; u++) {
        const long long i = base + u * 256;
        if (i < n) __stcs(out + i, __ldg(vals + p[u]));
    }
}

// Work items (H3): one item = up to ITEM3 consecutive records of ONE group in the (group, M)-ordered stream, so that
// a thread block shares every loop bound, table row and the group's slab.  One thread per group (plus one for the
// bucket of the requests failing S1-S6): the group's records are the buckets [gbase[g], gbase[g+1]).  `bounds[b]` is
// the END of bucket b after the scatter (ends = 1: the cursor array) or its START for pre-sorted input (ends = 0: the
// scanned histogram).  item = {first position, records, group | ZERO_ITEM, first isospin bin | bins << 8}: a group
// whose 20 isospin-combined slabs exceed one stage (VW_WORDS) is evaluated in rounds over bin ranges, one item per
// (chunk, round); a record is evaluated by the round that holds its bin.
// Groups with at most SMALL_ITEM3 records go to a second list (filled from the END of the item array, counted in
// n_items[1]): a single warp evaluates them directly from the five isospin planes (k_transform3_small).  Groups whose
// slab does not fit a stage even four bins at a time (gsize > 639: no such group in the five workloads, but tuples
// of three j = 15/2 orbitals have one) go to the same list in chunks of SMALL_ITEM3 records: that path has no
// capacity limit.
// 16: measured optimum (64 -> 16: config 3 at 2^22 requests 619 -> 551 us, config 4 batch of 2^24 2.64 -> 2.49 ms, config 3 at
// 2^26 unchanged; 8: same; 4: worse) -- the staged kernel amortises its slab copy from about 16 records on
constexpr uint32_t SMALL_ITEM3 = 16;
__device__ __forceinline__ uint32_t bins_per_round3(uint32_t gsize, int f32)
{
    const uint32_t b = ((uint32_t)VW_WORDS / vw_stride(gsize, f32)) & ~3u;   // multiple of 4: every round starts 16-byte aligned
    return min(b, (uint32_t)NBIN3);
}
// dense_tau < 0: no group takes the dense-block path (H5'); otherwise a feasible group does if its records number at
// least dense_tau * (its (bra, ket) m-state pairs with equal M) -- 0 = every feasible group (MFDN_FORCE_DENSE).  Such a
// group gets one entry per non-empty (group, M) bucket in `ditems` {first position, records, group, index of M}.
__global__ void __launch_bounds__(256) k_items3(const uint32_t* __restrict__ bounds, const uint32_t* __restrict__ gbase,
                                               uint32_t n_groups, uint32_t n_buckets, int ends, uint32_t n,
                                               const uint4* __restrict__ sgrp, uint4* __restrict__ items, uint32_t last_slot,
                                               uint32_t* __restrict__ n_items, float dense_tau, uint4* __restrict__ ditems, int vw_f32)
{
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;   // g == n_groups: the bucket of the invalid requests
    uint32_t start = 0, end = 0, gsize = 0, b0 = 0, b1 = 0;
    bool zero = true, dense = false;
    if (g <= n_groups) {
        b0 = g < n_groups ? __ldg(gbase + g) : n_buckets - 1u;
        b1 = g < n_groups ? __ldg(gbase + g + 1) : n_buckets;
        if (b1 > b0) {
            if (ends) { start = b0 ? bounds[b0 - 1] : 0u; end = bounds[b1 - 1]; }
            else { start = bounds[b0]; end = b1 < n_buckets ? bounds[b1] : n; }
        }
        if (end > start && g < n_groups) {
            const uint4 sg = __ldg(sgrp + g);
            zero = sg.x == NO_SLAB;
            gsize = sg.y;
            dense = !zero && dense_tau >= 0.f && (sg.w >> 31) && (float)(end - start) >= dense_tau * (float)(sg.w & 0x7FFFFFFFu);
        }
    }
    if (dense) {   // one entry per non-empty bucket; the group is left out of the two lists below
        for (uint32_t b = b0; b < b1; b++) {
            const uint32_t s0 = ends ? (b ? bounds[b - 1] : 0u) : bounds[b];
            const uint32_t s1 = ends ? bounds[b] : (b + 1 < n_buckets ? bounds[b + 1] : n);
            if (s1 > s0) ditems[atomicAdd(n_items + 2, 1u)] = make_uint4(s0, s1 - s0, g, b - b0);
        }
        start = end = 0;
    }
    const uint32_t cnt = end - start;
    const uint32_t bpr = zero ? (uint32_t)NBIN3 : bins_per_round3(gsize, vw_f32);
    const bool small = cnt <= SMALL_ITEM3 || bpr == 0u;
    const uint32_t rounds = small ? 0u : (NBIN3 + bpr - 1u) / bpr;
    const uint32_t k = small ? 0u : ((cnt + ITEM3 - 1) / ITEM3) * rounds, ks = small ? (cnt + SMALL_ITEM3 - 1) / SMALL_ITEM3 : 0u;
    // warp-aggregated append: the lists stay (nearly) in group order, neighbours share the bra tuple's tables
    const int lane = threadIdx.x & 31;
    uint32_t incl = k, incs = ks;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        uint32_t x = __shfl_up_sync(0xFFFFFFFFu, incl, off), y = __shfl_up_sync(0xFFFFFFFFu, incs, off);
        if (lane >= off) { incl += x; incs += y; }
    }
    uint32_t base = 0, bases = 0;
    if (lane == 31 && incl) base = atomicAdd(n_items, incl);
    if (lane == 31 && incs) bases = atomicAdd(n_items + 1, incs);
    base = __shfl_sync(0xFFFFFFFFu, base, 31);
    bases = __shfl_sync(0xFFFFFFFFu, bases, 31);
    if (cnt == 0) return;
    const uint32_t gz = zero ? ZERO_ITEM : g;
    if (small) {
        uint32_t slot = last_slot - (bases + incs - ks);
        for (uint32_t j = 0; j * SMALL_ITEM3 < cnt; j++) items[slot--] = make_uint4(start + j * SMALL_ITEM3, min(SMALL_ITEM3, cnt - j * SMALL_ITEM3), gz, 0u);
        return;
    }
    uint32_t slot = base + incl - k;
    for (uint32_t j = 0; j * ITEM3 < cnt; j++)
        for (uint32_t r = 0; r < rounds; r++)
            items[slot++] = make_uint4(start + j * ITEM3, min((uint32_t)ITEM3, cnt - j * ITEM3), gz, (r * bpr) | (min(bpr, NBIN3 - r * bpr) << 8));
}

// H3-H6 for small groups: one warp per item.  The group's loop bounds, table rows and slab addresses are warp-uniform, the
// lanes differ in their projections (sigma) and isospin bin.  Same operations in the same order as the staged path of
// k_transform3 (Vw of the record's bin from the isospin-combined slabs, then ck, then cb, then the sum over J in ascending
// order), so a request's value does not depend on which of the two kernels its group happened to go to.
// A warp is PARTS sub-warps of 32 / PARTS lanes: lane = (record r, part p).  Part p evaluates the J blocks q = p, p + PARTS, ..
// of its record; the PARTS blocks of a round run side by side under the largest bounds of the round (neighbouring J have
// similar ranges), the block sums are then added in ascending J by every lane (shuffles), which keeps the summation
// order of the one-lane-per-record form.  Groups of at most SMALL_SPLIT records (config 4: a 2^24-request batch leaves
// about 6 records per group of its uniform part) take PARTS = 4, eight records per pass; larger ones PARTS = 1.
constexpr uint32_t SMALL_SPLIT = 24;
template <int PARTS, bool F32>
__device__ __forceinline__ void small_group3(const Tables& T, uint32_t pos0, uint32_t cnt, int nblk, int2 ib_l, int2 ik_l, uint32_t voff_l,
                                             uint32_t tb_off, uint32_t tk_off, const uint32_t* __restrict__ vw, uint32_t gsize,
                                             const unsigned long long* __restrict__ recs, double* __restrict__ out, int lane)
{
    constexpr int W = 32 / PARTS;
    const int r = lane % W, p = lane / W;
    const double* __restrict__ dtab = T.dtab3;
    const uint32_t S = vw_stride(gsize, F32);
    for (uint32_t r0 = 0; r0 < cnt; r0 += W) {
        const bool valid = r0 + r < cnt;
        const uint32_t lo = (uint32_t)__ldg(recs + pos0 + (valid ? r0 + r : r0));
        const uint32_t sb = lo & 0xFFFu, sk = (lo >> 12) & 0xFFFu;
        const uint32_t* __restrict__ vwl = vw + (size_t)((lo >> 24) & 31u) * S;   // low words of the record's bin; high words gsize further
        double total = 0.0;
        for (int q0 = 0; q0 < nblk; q0 += PARTS) {
            const int q = q0 + p;
            const bool has = q < nblk;
            const int src = has ? q : 0;
            const uint32_t ibx = (uint32_t)__shfl_sync(0xFFFFFFFFu, ib_l.x, src), ikx = (uint32_t)__shfl_sync(0xFFFFFFFFu, ik_l.x, src);
            int nb = __shfl_sync(0xFFFFFFFFu, ib_l.y, src), nk = __shfl_sync(0xFFFFFFFFu, ik_l.y, src);
            uint32_t c = __shfl_sync(0xFFFFFFFFu, voff_l, src);
            if (!has || nk <= 0) nb = 0;
            int nbmax = nb, nkmax = nb > 0 ? nk : 0;
            if (PARTS > 1) {
#pragma unroll
                for (int off = W; off < 32; off <<= 1) {
                    nbmax = max(nbmax, __shfl_xor_sync(0xFFFFFFFFu, nbmax, off));
                    nkmax = max(nkmax, __shfl_xor_sync(0xFFFFFFFFu, nkmax, off));
                }
            }
            const uint32_t P = (uint32_t)row_pitch3(nk);
            const double* __restrict__ cbp = dtab + (tb_off + ibx + sb * (uint32_t)nb);
            const double* __restrict__ ckp = dtab + (tk_off + ikx + sk * (uint32_t)nk);
            double t = 0.0;
            for (int i = 0; i < nbmax; i++) {
                const bool row = i < nb;
                const double cb = row ? __ldg(cbp + i) : 0.0;
                double acc = 0.0;
                for (int k0 = 0; k0 < nkmax; k0 += 4) {   // four cells' loads (12) in flight before the first multiply
                    double ck[4], v[4];
#pragma unroll
                    for (int u = 0; u < 4; u++) {
                        const bool on = row && k0 + u < nk;
                        const uint32_t cell = on ? c + (uint32_t)(k0 + u) : 0u;
                        ck[u] = on ? __ldg(ckp + k0 + u) : 0.0;
                        const uint32_t lw = on ? __ldg(vwl + cell) : 0u, hw = (on && !F32) ? __ldg(vwl + gsize + cell) : 0u;
                        v[u] = F32 ? (double)__uint_as_float(lw) : __hiloint2double((int)hw, (int)lw);
                    }
#pragma unroll
                    for (int u = 0; u < 4; u++)
                        if (row && k0 + u < nk) acc = (k0 + u) ? fma(ck[u], v[u], acc) : ck[u] * v[u];
                }
                if (row) { t = fma(cb, acc, t); c += P; }
            }
            if (PARTS > 1) {
#pragma unroll
                for (int pp = 0; pp < PARTS; pp++) {
                    const double tt = __shfl_sync(0xFFFFFFFFu, t, pp * W + r);
                    if (q0 + pp < nblk) total += tt;
                }
            } else {
                total += t;
            }
        }
        if (valid && p == 0) out[pos0 + r0 + r] = (((lo >> 29) & 1u) ? -total : total) + 0.0;   // + 0.0: never store -0
    }
}

template <bool F32>
__global__ void __launch_bounds__(128) k_transform3_small(Tables T, const uint4* __restrict__ items, uint32_t last_slot,
                                                          const uint32_t* __restrict__ n_items_p,
                                                          const unsigned long long* __restrict__ recs, double* __restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    const uint32_t n_small = __ldg(n_items_p + 1);
    const uint32_t nt = (uint32_t)T.n_tup3;
    for (uint32_t it = gw; it < n_small; it += nw) {
        const uint4 item = __ldg(items + (last_slot - it));
        const uint32_t pos0 = item.x, cnt = item.y, g = item.z;
        if (g == ZERO_ITEM) {
            for (uint32_t r = lane; r < cnt; r += 32) out[pos0 + r] = 0.0;
            continue;
        }
        const uint32_t tb = g / nt, tk = g - tb * nt;
        const int4 kb = __ldg(T.tk3 + tb), kk = __ldg(T.tk3 + tk);
        const uint4 sg = __ldg(T.sgrp3 + g);
        const int Jminb = (kb.w >> 16) & 255, Jmink = (kk.w >> 16) & 255;
        const int Jlo = max(Jminb, Jmink), Jhi = min((kb.w >> 24) & 255, (kk.w >> 24) & 255);
        const int nblk = ((Jhi - Jlo) >> 1) + 1;
        // lane q holds the J block q: {offset in the tuple's coefficient table, rows} of either side, first Vw cell
        int2 ib = make_int2(0, 0), ik = make_int2(0, 0);
        if (lane < nblk) {
            ib = __ldg(T.jinfo3 + kb.z + ((Jlo - Jminb) >> 1) + lane);
            ik = __ldg(T.jinfo3 + kk.z + ((Jlo - Jmink) >> 1) + lane);
        }
        const uint32_t vv = (uint32_t)(ib.y * row_pitch3(ik.y));
        uint32_t iv = vv;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const uint32_t x = __shfl_up_sync(0xFFFFFFFFu, iv, off);
            if (lane >= off) iv += x;
        }
        const uint32_t* __restrict__ vw = T.vw20 + (size_t)sg.z * 4;
        if (cnt <= SMALL_SPLIT) small_group3<4, F32>(T, pos0, cnt, nblk, ib, ik, iv - vv, (uint32_t)kb.x, (uint32_t)kk.x, vw, sg.y, recs, out, lane);
        else small_group3<1, F32>(T, pos0, cnt, nblk, ib, ik, iv - vv, (uint32_t)kb.x, (uint32_t)kk.x, vw, sg.y, recs, out, lane);
    }
}

// ------------------------------------------------------------------------------- H3-H6, pipelined transform
// mbarrier / bulk-copy (TMA, 1-D) primitives
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* b, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* b)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory");
}
__device__ __forceinline__ void mbar_arrive_tx(unsigned long long* b, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(b)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* b, uint32_t parity)
{
    const uint32_t a = smem_u32(b);
    uint32_t ok;
    do {
        // the last operand lets the hardware suspend the warp until the phase completes (or the time hint, ns, runs out)
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(a), "r"(parity), "r"(1000000u) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, unsigned long long* b)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(b)) : "memory");
}

#ifndef MFDN_TR_CW
#define MFDN_TR_CW 4
#endif
#ifndef MFDN_TR_SLOTS
#define MFDN_TR_SLOTS 8
#endif
#ifndef MFDN_TR_MINB
#define MFDN_TR_MINB 4
#endif
#ifndef MFDN_TR_RING
#define MFDN_TR_RING 9216
#endif
#ifndef MFDN_TR_PF
#define MFDN_TR_PF 0
#endif
constexpr int TR_CW = MFDN_TR_CW;               // consumer warps per block
constexpr int TR_THREADS = (TR_CW + 1) * 32;    // + one producer warp
constexpr int TR_SLOTS = MFDN_TR_SLOTS;         // work items in flight per block
constexpr int MAX_JBLK = 32;                    // common J values of a group (2J <= 63)
constexpr int BATCH3 = 64;                      // records per consumer-warp batch (two per lane)
constexpr int REC_WORDS_MAX = (ITEM3 + 2) * 2;  // records are copied from an even position: one record of slack at either end
// Ring of 32-bit words holding, per work item in flight, everything its consumer warps read: the isospin-combined slabs
// and the records (both landed by bulk copies) and the J-block descriptors (written by the producer warp).  At least
// one item of maximal size; typical items (4 KB of slabs, 3 KB of records) leave room for five in flight.  A small ring
// keeps more of the SM's 228 KB as L1 for the coefficient tables (ncu: with two fixed 25 KB stages per block the L1 hit
// rate of the coefficient gathers was 60 %).  Swept with the items handed out dynamically (pre-sorted call of config 3 /
// one batch of config 4, ms): 6656 words 2.053 / 2.142, 7424 2.033, 8192 2.034 / 2.095, 9216 2.025, 10240 2.043 / 2.067.
constexpr int RING_WORDS = MFDN_TR_RING;
static_assert(RING_WORDS >= VW_WORDS + REC_WORDS_MAX + MAX_JBLK * 4, "ring must hold one maximal work item");
enum { SC_POS0, SC_CNT, SC_GROUP, SC_SB, SC_SK, SC_PB0, SC_PK0, SC_JINFO, SC_GSIZE, SC_STRIDE, SC_BINS, SC_ROFF, SC_VW, SC_REC, SC_DESC, SC_NEXT };
struct __align__(16) Pipe3 {
    uint32_t ring[RING_WORDS];
    uint32_t sc[TR_SLOTS][16];                  // item scalars, see SC_* (SC_VW, SC_REC, SC_DESC: ring offsets in words)
    unsigned long long full[TR_SLOTS], empty[TR_SLOTS];
    uint32_t start_of[TR_SLOTS];                // ring offset of the item in each slot (producer's bookkeeping)
};

// one Vw value from its two staged 32-bit words: `lo` / `hi` are shared-space byte addresses of word 0 of the low / high plane
// of the record's bin, OFF the compile-time word offset of the cell
// F32 (fp32-stored slabs, MFDN_OPT_SLAB_FP32): one word per value at `lo`, widened to fp64; `hi` is unused
template <int OFF, bool F32>
__device__ __forceinline__ double ldvw(uint32_t lo, uint32_t hi)
{
    if constexpr (F32) {
        float f;
        asm("ld.shared.f32 %0, [%1+%2];" : "=f"(f) : "r"(lo), "n"(OFF * 4));
        return (double)f;
    }
    uint32_t a, b;
    asm("ld.shared.u32 %0, [%1+%2];" : "=r"(a) : "r"(lo), "n"(OFF * 4));
    asm("ld.shared.u32 %0, [%1+%2];" : "=r"(b) : "r"(hi), "n"(OFF * 4));
    return __hiloint2double((int)b, (int)a);
}

// N consecutive coefficients of one m-state in a J block (16-byte aligned when N is even)
template <int N>
__device__ __forceinline__ void ldcoef(const double* __restrict__ p, double (&c)[N])
{
    if constexpr (N % 2 == 0) {
#pragma unroll
        for (int i = 0; i < N / 2; i++) {
            const double2 v = __ldg(reinterpret_cast<const double2*>(p) + i);
            c[2 * i] = v.x;
            c[2 * i + 1] = v.y;
        }
    } else {
#pragma unroll
        for (int i = 0; i < N; i++) c[i] = __ldg(p + i);
    }
}

// One J block of the sum for TWO records of the group (A and B, 32 stream positions apart):
//   sum_i cb(i) * sum_k ck(k) * Vw[i][k],   cb = bq[sigma_b * nb + i],  ck = kq[sigma_k * nk + k]
// (bq, kq: the J block of the bra / ket tuple's coefficient table), Vw rows (padded to even length) read from the staged
// word planes at vi + i * P + k.  Bra and ket range sizes known at compile time: every load of the block is issued before
// the first multiply, the loop control is shared by the two records.
template <int NB, int NK, int I, bool F32>
__device__ __forceinline__ void vw_row(uint32_t lo, uint32_t hi, double (&v)[NK])
{
    constexpr int P = (NK + 1) & ~1;
    if constexpr (NK >= 1) v[0] = ldvw<I * P + 0, F32>(lo, hi);
    if constexpr (NK >= 2) v[1] = ldvw<I * P + 1, F32>(lo, hi);
    if constexpr (NK >= 3) v[2] = ldvw<I * P + 2, F32>(lo, hi);
    if constexpr (NK >= 4) v[3] = ldvw<I * P + 3, F32>(lo, hi);
    if constexpr (NK >= 5) v[4] = ldvw<I * P + 4, F32>(lo, hi);
    if constexpr (NK >= 6) v[5] = ldvw<I * P + 5, F32>(lo, hi);
    if constexpr (NK >= 7) v[6] = ldvw<I * P + 6, F32>(lo, hi);
    if constexpr (NK >= 8) v[7] = ldvw<I * P + 7, F32>(lo, hi);
}
template <int NB, int NK, int I, bool F32>
__device__ __forceinline__ void j_rows(const double (&ckA)[NK], const double (&ckB)[NK], const double (&cbA)[NB], const double (&cbB)[NB],
                                       uint32_t loA, uint32_t hiA, uint32_t loB, uint32_t hiB, double& tA, double& tB)
{
    if constexpr (I < NB) {
        double vA[NK], vB[NK];
        vw_row<NB, NK, I, F32>(loA, hiA, vA);
        vw_row<NB, NK, I, F32>(loB, hiB, vB);
        double accA = ckA[0] * vA[0], accB = ckB[0] * vB[0];
#pragma unroll
        for (int k = 1; k < NK; k++) {
            accA = fma(ckA[k], vA[k], accA);
            accB = fma(ckB[k], vB[k], accB);
        }
        tA = fma(cbA[I], accA, tA);
        tB = fma(cbB[I], accB, tB);
        j_rows<NB, NK, I + 1, F32>(ckA, ckB, cbA, cbB, loA, hiA, loB, hiB, tA, tB);
    }
}
// boff / koff: offsets (doubles) of the J block in the bra / ket tuple's coefficient table; loA.. : shared-space byte addresses
// of the block's first Vw cell in the low / high word plane of record A's / B's bin
template <int NB, int NK, bool F32>
__device__ __forceinline__ void j_block3x2(const double* __restrict__ dtab, uint32_t boff, uint32_t koff, uint32_t sbA,
                                           uint32_t skA, uint32_t sbB, uint32_t skB, uint32_t loA, uint32_t hiA, uint32_t loB, uint32_t hiB,
                                           double& totA, double& totB)
{
    double ckA[NK], ckB[NK], cbA[NB], cbB[NB];
    ldcoef<NK>(dtab + (koff + skA * NK), ckA);
    ldcoef<NK>(dtab + (koff + skB * NK), ckB);
    ldcoef<NB>(dtab + (boff + sbA * NB), cbA);
    ldcoef<NB>(dtab + (boff + sbB * NB), cbB);
    double tA = 0.0, tB = 0.0;
    j_rows<NB, NK, 0, F32>(ckA, ckB, cbA, cbB, loA, hiA, loB, hiB, tA, tB);
    totA += tA;
    totB += tB;
}
// The same with a run-time loop over the bra rows (blocks with more than 4 rows or columns, NK <= 8)
template <int NK, bool F32>
__device__ __forceinline__ void j_block3x2_rows(const double* __restrict__ dtab, uint32_t boff, uint32_t koff, uint32_t sbA,
                                                uint32_t skA, uint32_t sbB, uint32_t skB, int nb, uint32_t loA, uint32_t hiA, uint32_t loB,
                                                uint32_t hiB, double& totA, double& totB)
{
    constexpr int P = (NK + 1) & ~1;
    double ckA[NK], ckB[NK];
    ldcoef<NK>(dtab + (koff + skA * NK), ckA);
    ldcoef<NK>(dtab + (koff + skB * NK), ckB);
    const double* __restrict__ bA = dtab + (boff + sbA * (uint32_t)nb);
    const double* __restrict__ bB = dtab + (boff + sbB * (uint32_t)nb);
    double tA = 0.0, tB = 0.0;
#pragma unroll 2
    for (int i = 0; i < nb; i++) {
        const double cbA = __ldg(bA + i), cbB = __ldg(bB + i);
        double vA[NK], vB[NK];
        vw_row<1, NK, 0, F32>(loA, hiA, vA);
        vw_row<1, NK, 0, F32>(loB, hiB, vB);
        loA += P * 4; hiA += P * 4; loB += P * 4; hiB += P * 4;
        double accA = ckA[0] * vA[0], accB = ckB[0] * vB[0];
#pragma unroll
        for (int k = 1; k < NK; k++) {
            accA = fma(ckA[k], vA[k], accA);
            accB = fma(ckB[k], vB[k], accB);
        }
        tA = fma(cbA, accA, tA);
        tB = fma(cbB, accB, tB);
    }
    totA += tA;
    totB += tB;
}

// any ket range size (nk > 8): ket coefficient re-read per cell
__device__ __noinline__ double j_block3_generic(const double* __restrict__ bp, const double* __restrict__ kp, int nb, int nk, uint32_t lo,
                                                uint32_t hi, bool f32)
{
    const int P = row_pitch3(nk);
    double total = 0.0;
    for (int i = 0; i < nb; i++) {
        const double cb = __ldg(bp + i);
        double acc = 0.0;
        for (int k = 0; k < nk; k++) {
            uint32_t a, b = 0u;
            asm("ld.shared.u32 %0, [%1];" : "=r"(a) : "r"(lo + 4u * k));
            if (!f32) asm("ld.shared.u32 %0, [%1];" : "=r"(b) : "r"(hi + 4u * k));
            const double ck = __ldg(kp + k), v = f32 ? (double)__uint_as_float(a) : __hiloint2double((int)b, (int)a);
            acc = k ? fma(ck, v, acc) : ck * v;
        }
        total = fma(cb, acc, total);
        lo += 4u * P; hi += 4u * P;
    }
    return total;
}

// H3-H6.  Persistent blocks walk the item list (item k of a block = list entry blockIdx.x + k * gridDim.x) with up to
// TR_SLOTS items in flight:
//  * the PRODUCER warp, per item: reads the group's descriptors, reserves room in the block's shared-memory ring (FIFO;
//    it waits for the oldest items to be released when the ring or the slot table is full), builds the J-block table
//    (bounds of the three nested loops of PAPER.md:61, shared by every record of the group) and starts two bulk copies
//    (cp.async.bulk -> UBLKCP, completion on the slot's mbarrier): the group's isospin-combined slabs Vw[bin][cell] and
//    the item's records.  It never touches the data itself, so it runs several items ahead of the consumers and every
//    global latency of the prologue is off their critical path;
//  * the CONSUMER warps wait for the slot, then take every TR_CW-th batch of 64 records (two per lane, stream order).  The stream
//    is ordered by (group, M) and the coefficient tables are M-major: the lanes of a warp read one or two cache lines
//    per coefficient on the bra AND on the ket side.  Every lane evaluates
//        sum_J sum_J12 cb(J12,J) sum_J12' ck(J12',J) Vw[bin][J,J12,J12']
//    for its records with warp-uniform loop bounds (first J block = the smallest |M| in the warp; coefficients are 0
//    for J < |M|), and stores the signed value at the record's stream position (coalesced).
// No block-wide barrier after the prologue.
template <bool F32>
__global__ void __launch_bounds__(TR_THREADS, MFDN_TR_MINB) k_transform3(Tables T, const uint4* __restrict__ items, const uint32_t* __restrict__ n_items_p,
                                                                     const unsigned long long* __restrict__ recs, double* __restrict__ out,
                                                                     uint32_t* __restrict__ next_item)
{
    __shared__ Pipe3 P;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) {
        for (int s = 0; s < TR_SLOTS; s++) { mbar_init(&P.full[s], 1u); mbar_init(&P.empty[s], (uint32_t)TR_CW); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    const uint32_t n_items = __ldg(n_items_p);
    const uint32_t nt = (uint32_t)T.n_tup3;
    if (warp == TR_CW) {
        // ------------------------------------------------------------------ producer (all lanes run the same control flow)
        uint32_t k = 0, rel = 0, head = 0;       // items issued, items released (FIFO), next free ring word
        // The descriptor loads of an item form a chain of three dependent global loads (list entry -> tuple and group
        // descriptors -> J-block rows).  They are software-pipelined over the item loop: every load is issued one full
        // iteration before its result is used, so the producer's time per item is one slot hand-over, not three L2 latencies
        // (ncu: consumers spent 11 % of their samples waiting on `full` behind short items).
        struct D1 { int4 kb, kk; uint4 sg; };
        struct D2 { int2 jb, jk; int gJlo, gnblk; };
        auto ld_item = [&](uint32_t it) { return it < n_items ? __ldg(items + it) : make_uint4(0u, 0u, ZERO_ITEM, 0u); };
        auto ld_d1 = [&](const uint4& item) {
            D1 d{make_int4(0, 0, 0, 0), make_int4(0, 0, 0, 0), make_uint4(0u, 0u, 0u, 0u)};
            if (item.z != ZERO_ITEM) {
                const uint32_t tb = item.z / nt, tk = item.z - tb * nt;
                d.kb = __ldg(T.tk3 + tb);
                d.kk = __ldg(T.tk3 + tk);
                d.sg = __ldg(T.sgrp3 + item.z);
            }
            return d;
        };
        auto ld_d2 = [&](const uint4& item, const D1& d) {
            D2 e{make_int2(0, 0), make_int2(0, 0), 0, 0};
            if (item.z != ZERO_ITEM) {
                const int Jminb = (d.kb.w >> 16) & 255, Jmink = (d.kk.w >> 16) & 255;
                e.gJlo = max(Jminb, Jmink);
                e.gnblk = ((min((d.kb.w >> 24) & 255, (d.kk.w >> 24) & 255) - e.gJlo) >> 1) + 1;
                if (lane < e.gnblk) {
                    e.jb = __ldg(T.jinfo3 + d.kb.z + ((e.gJlo - Jminb) >> 1) + lane);
                    e.jk = __ldg(T.jinfo3 + d.kk.z + ((e.gJlo - Jmink) >> 1) + lane);
                }
            }
            return e;
        };
        // Items are handed out through a global counter (one atomic per item, claimed one iteration before its value is used):
        // with a fixed round-robin share the blocks finished up to 4 % apart (ncu: warps active 29.9 % of peak against 31.25 % for
        // 20 resident warps), now the tail is one item.
        auto claim = [&]() { uint32_t v = 0u; if (lane == 0) v = atomicAdd(next_item, 1u); return v; };   // valid in lane 0
        auto bcast = [&](uint32_t v) { return __shfl_sync(0xFFFFFFFFu, v, 0); };
        uint32_t it = bcast(claim()), it1 = bcast(claim()), it2 = bcast(claim()), raw3 = claim();
        uint4 item = ld_item(it), item1 = ld_item(it1), item2 = ld_item(it2);
        D1 d0 = ld_d1(item), d1 = ld_d1(item1);
        D2 e0 = ld_d2(item, d0);
        for (; it < n_items; k++) {
            const uint32_t s = k % TR_SLOTS;
            // loads for the items behind this one
            const uint32_t it3 = bcast(raw3);
            raw3 = claim();
            const uint4 item3 = ld_item(it3);
            it = it1; it1 = it2; it2 = it3;
            const D1 d2 = ld_d1(item2);
            const D2 e1 = ld_d2(item1, d1);
            const uint4 cur = item;
            const int4 kb = d0.kb, kk = d0.kk;
            const uint4 sg = d0.sg;
            const int2 jb = e0.jb, jk = e0.jk;
            const int gnblk = e0.gnblk, gJlo = e0.gJlo;
            item = item1; item1 = item2; item2 = item3;
            d0 = d1; d1 = d2;
            e0 = e1;
            const uint32_t pos0 = cur.x, cnt = cur.y, g = cur.z;
            const bool zero = g == ZERO_ITEM;
            const uint32_t gsize = sg.y, S = vw_stride(gsize, F32), bin_lo = cur.w & 255u, bins = cur.w >> 8;
            const uint32_t vw_words = zero ? 0u : (bins * S + 3u) & ~3u;
            const uint32_t rec_words = zero ? 0u : (((pos0 & 1u) + cnt + 1u) & ~1u) * 2u;
            const uint32_t need = vw_words + rec_words + (uint32_t)gnblk * 4u;
            // reserve `need` contiguous words: the live region is [start_of[rel], head), possibly wrapped
            uint32_t at;
            for (;;) {
                bool ok = false;
                at = head;
                if (k - rel < (uint32_t)TR_SLOTS) {
                    if (rel == k) { at = 0u; ok = true; }     // nothing in flight
                    else {
                        const uint32_t tail = P.start_of[rel % TR_SLOTS];
                        if (head > tail) {
                            if (head + need <= (uint32_t)RING_WORDS) ok = true;
                            else if (need < tail) { at = 0u; ok = true; }
                        } else if (head + need < tail) ok = true;
                    }
                }
                if (ok) break;
                mbar_wait(&P.empty[rel % TR_SLOTS], (rel / TR_SLOTS) & 1u);   // every consumer warp has left the oldest item
                rel++;
            }
            head = at + need;
            if (lane == 0) P.start_of[s] = at;
            __syncwarp();
            uint32_t* sc = P.sc[s];
            if (zero) {
                if (lane == 0) {
                    sc[SC_POS0] = pos0; sc[SC_CNT] = cnt; sc[SC_GROUP] = ZERO_ITEM;
                    mbar_arrive(&P.full[s]);
                }
                continue;
            }
            // exclusive prefix sum of the Vw cells over the J blocks
            const uint32_t rb = (uint32_t)jb.y, rk = (uint32_t)jk.y, vv = (uint32_t)(jb.y * row_pitch3(jk.y));
            uint32_t iv = vv;
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                uint32_t xv = __shfl_up_sync(0xFFFFFFFFu, iv, off);
                if (lane >= off) iv += xv;
            }
            const uint32_t o_vw = at, o_rec = at + vw_words, o_desc = o_rec + rec_words;
            if (lane < gnblk) {
                // dispatch code: 0..15 fully unrolled (nb, nk <= 4); 16 + nk row-loop templates (nk <= 8); 25 generic
                const uint32_t code = (rb - 1u < 4u && rk - 1u < 4u) ? (rb - 1u) * 4u + (rk - 1u) : (rk - 1u < 8u && rb > 0u) ? 16u + rk : 25u;
                *reinterpret_cast<uint4*>(&P.ring[o_desc + 4u * lane]) =
                    make_uint4(rb | (rk << 8) | (code << 16), (uint32_t)kb.x + (uint32_t)jb.x, (uint32_t)kk.x + (uint32_t)jk.x, iv - vv);
            }
            if (lane == 0) {
                sc[SC_POS0] = pos0; sc[SC_CNT] = cnt; sc[SC_GROUP] = g;
                sc[SC_SB] = 0u; sc[SC_SK] = 0u; sc[SC_PB0] = 0u; sc[SC_PK0] = 0u;
                sc[SC_JINFO] = ((uint32_t)kb.w & 0xFFu) | ((uint32_t)gJlo << 8) | ((uint32_t)gnblk << 16);
                sc[SC_GSIZE] = gsize; sc[SC_STRIDE] = S; sc[SC_BINS] = cur.w; sc[SC_ROFF] = pos0 & 1u;
                sc[SC_VW] = o_vw; sc[SC_REC] = o_rec; sc[SC_DESC] = o_desc;
            }
            __syncwarp();
            if (lane == 0) {
                mbar_arrive_tx(&P.full[s], (vw_words + rec_words) * 4u);
                bulk_g2s(&P.ring[o_vw], T.vw20 + (size_t)sg.z * 4 + (size_t)bin_lo * S, vw_words * 4u, &P.full[s]);
                bulk_g2s(&P.ring[o_rec], recs + (pos0 & ~1u), rec_words * 4u, &P.full[s]);
            }
        }
        // no items left: tell the consumers (the slot of entry k is free once item k - TR_SLOTS has been released)
        while (k - rel >= (uint32_t)TR_SLOTS) {
            mbar_wait(&P.empty[rel % TR_SLOTS], (rel / TR_SLOTS) & 1u);
            rel++;
        }
        if (lane == 0) {
            uint32_t* sc = P.sc[k % TR_SLOTS];
            sc[SC_POS0] = 0u; sc[SC_CNT] = 0u; sc[SC_GROUP] = STOP_ITEM;
            mbar_arrive(&P.full[k % TR_SLOTS]);
        }
        return;
    }
    // ---------------------------------------------------------------------- consumers
    const double* __restrict__ dtab = T.dtab3;
    for (uint32_t k = 0;; k++) {
        const uint32_t s = k % TR_SLOTS;
        uint32_t* sc = P.sc[s];
        mbar_wait(&P.full[s], (k / TR_SLOTS) & 1u);
        const uint4 s0 = *reinterpret_cast<const uint4*>(&sc[0]);    // pos0, cnt, group, -
        if (s0.z == STOP_ITEM) break;
        const uint32_t pos0 = s0.x, cnt = s0.y;
        if (s0.z == ZERO_ITEM) {
            for (uint32_t b = ((uint32_t)warp + k) % TR_CW * BATCH3; b < cnt; b += TR_CW * BATCH3) {
                if (b + lane < cnt) out[pos0 + b + lane] = 0.0;
                if (b + 32 + lane < cnt) out[pos0 + b + 32 + lane] = 0.0;
            }
        } else {
            const uint4 s1 = *reinterpret_cast<const uint4*>(&sc[4]);    // -, -, -, jinfo
            const uint4 s2 = *reinterpret_cast<const uint4*>(&sc[8]);    // gsize, stride, bins, roff
            const uint4 s3 = *reinterpret_cast<const uint4*>(&sc[12]);   // ring offsets: vw, rec, desc
            const uint32_t G = s2.x, S = s2.y, bin_lo = s2.z & 255u, bins = s2.z >> 8;
            const int sumj = s1.w & 255, Jlo = (s1.w >> 8) & 255, nblk = (int)(s1.w >> 16);
            const unsigned long long* irec = reinterpret_cast<const unsigned long long*>(&P.ring[s3.y]) + s2.w;
            const uint32_t vw0 = smem_u32(&P.ring[s3.x]), G4 = G * 4u;
            const uint4* desc = reinterpret_cast<const uint4*>(&P.ring[s3.z]);
            // batches of the item are dealt round-robin to the warps, starting with a different warp for every item (a shared
            // counter claimed with an atomic cost a shared-memory atomic + shuffle round trip per batch: 4.13 -> 4.05 ms per step)
            for (uint32_t base = ((uint32_t)warp + k) % TR_CW * BATCH3; base < cnt; base += TR_CW * BATCH3) {
                // lane l takes stream positions base+l (A) and base+32+l (B); lanes past the end of the item redo its last
                // record and skip the store
                const uint32_t slotA = base + lane, slotB = slotA + 32u;
                const unsigned long long rcA = irec[min(slotA, cnt - 1u)], rcB = irec[min(slotB, cnt - 1u)];
                const uint32_t loA = (uint32_t)rcA, loB = (uint32_t)rcB;
                const uint32_t blA = ((loA >> 24) & 31u) - bin_lo, blB = ((loB >> 24) & 31u) - bin_lo;
                const int aMA = abs(2 * ((int)(rcA >> 30) & 63) - sumj), aMB = abs(2 * ((int)(rcB >> 30) & 63) - sumj);
                // first block with J >= |M| of any record of the warp (coefficients are 0 below a record's own |M|)
                const int q0 = max(0, ((int)__reduce_min_sync(0xFFFFFFFFu, (unsigned)min(aMA, aMB)) - Jlo + 1) >> 1);
                uint32_t sbA = loA & 0xFFFu, skA = (loA >> 12) & 0xFFFu, wA = vw0 + min(blA, bins - 1u) * S * 4u;
                uint32_t sbB = loB & 0xFFFu, skB = (loB >> 12) & 0xFFFu, wB = vw0 + min(blB, bins - 1u) * S * 4u;
                // opaque to the compiler: it then keeps these six values in registers across the J loop instead of re-deriving them
                // from the records in every block (30 of the 54 instructions of a block's dispatch were such re-derivations; -2.5 %)
                asm volatile("" : "+r"(sbA), "+r"(skA), "+r"(wA), "+r"(sbB), "+r"(skB), "+r"(wB));
                double totA = 0.0, totB = 0.0;
                for (int q = q0; q < nblk; q++) {
                    const uint4 d = desc[q];
                    const int nb = d.x & 255, nk = (d.x >> 8) & 255;
#if MFDN_TR_PF > 0
                    if (q + MFDN_TR_PF < nblk) {   // coefficient lines of a later J block on their way to L1 while this one is summed
                        const uint4 dn = desc[q + MFDN_TR_PF];
                        const uint32_t nbn = dn.x & 255u, nkn = (dn.x >> 8) & 255u;
                        asm volatile("prefetch.global.L1 [%0];" ::"l"(dtab + (dn.y + sbA * nbn)));
                        asm volatile("prefetch.global.L1 [%0];" ::"l"(dtab + (dn.z + skA * nkn)));
                        asm volatile("prefetch.global.L1 [%0];" ::"l"(dtab + (dn.y + sbB * nbn)));
                        asm volatile("prefetch.global.L1 [%0];" ::"l"(dtab + (dn.z + skB * nkn)));
                    }
#endif
                    const uint32_t vlA = wA + d.w * 4u, vlB = wB + d.w * 4u, vhA = vlA + G4, vhB = vlB + G4;
#define MFDN_BLK(NB, NK) case ((NB) - 1) * 4 + ((NK) - 1): j_block3x2<NB, NK, F32>(dtab, d.y, d.z, sbA, skA, sbB, skB, vlA, vhA, vlB, vhB, totA, totB); break;
#define MFDN_ROWS(NK) case 16 + (NK): j_block3x2_rows<NK, F32>(dtab, d.y, d.z, sbA, skA, sbB, skB, nb, vlA, vhA, vlB, vhB, totA, totB); break;
                    switch (d.x >> 16) {
                        MFDN_BLK(1, 1) MFDN_BLK(1, 2) MFDN_BLK(1, 3) MFDN_BLK(1, 4)
                        MFDN_BLK(2, 1) MFDN_BLK(2, 2) MFDN_BLK(2, 3) MFDN_BLK(2, 4)
                        MFDN_BLK(3, 1) MFDN_BLK(3, 2) MFDN_BLK(3, 3) MFDN_BLK(3, 4)
                        MFDN_BLK(4, 1) MFDN_BLK(4, 2) MFDN_BLK(4, 3) MFDN_BLK(4, 4)
                        MFDN_ROWS(1) MFDN_ROWS(2) MFDN_ROWS(3) MFDN_ROWS(4) MFDN_ROWS(5) MFDN_ROWS(6) MFDN_ROWS(7) MFDN_ROWS(8)
                        default: {
                            if (nk > 0 && nb > 0) {
                                totA += j_block3_generic(dtab + (d.y + sbA * (uint32_t)nb), dtab + (d.z + skA * (uint32_t)nk), nb, nk, vlA, vhA, F32);
                                totB += j_block3_generic(dtab + (d.y + sbB * (uint32_t)nb), dtab + (d.z + skB * (uint32_t)nk), nb, nk, vlB, vhB, F32);
                            }
                            break;
                        }
                    }
#undef MFDN_BLK
#undef MFDN_ROWS
                }
                // store unless past the end of the item or the bin belongs to another round; + 0.0: never store -0
                if (slotA < cnt && blA < bins) out[pos0 + slotA] = (((loA >> 29) & 1u) ? -totA : totA) + 0.0;
                if (slotB < cnt && blB < bins) out[pos0 + slotB] = (((loB >> 29) & 1u) ? -totB : totB) + 0.0;
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&P.empty[s]);
    }
}

// ------------------------------------------------------------------------------- H5': dense blocks on the fp64 tensor cores
// The block view A' = D^T A D (Fig. 1 at :69) for one (group, M) run and one isospin bin:
//     Vm[mu, mu'] = sum_{J >= |M|} sum_{J12, J12'} Cb[mu; J,J12] * Vw_bin[J; J12,J12'] * Ck[mu'; J,J12']
// over ALL bra m-states mu and ket m-states mu' of that M (the M-major order of the coefficient tables makes them index
// ranges), evaluated as two chained products:
//     T[mu, r] = sum_i Cb[mu; q(r), i] * Vw[q(r); i, k(r)]        r = flattened ket rows (J block q, J12' index k)
//     Vm       = T * Ck^T                                         8 x 8 tiles of mma.sync.m8n8k4.f64, K = r in chunks of 4
// One warp per run.  Per bin present in the run it fills Vm in its shared-memory buffer, then every record of that bin
// picks its entry.  T entries are computed directly in the A-fragment layout (lane = (mu, r mod 4)) and reused for all
// mu' tiles.  Pays only where most pairs of a block are requested (config 2, "ALL pairs"); see DESIGN.md for the
// measured break-even.  Summation order differs from the direct kernels: values agree to rounding, not bitwise.
constexpr int DN_WARPS = 4;
constexpr int DN_CHUNKS = DENSE_RMAX / 4;
struct DenseWarp3 {
    double vm[DENSE_CAP];
    uint4 rmap[DENSE_RMAX];   // per flattened ket row: {bra block offset, nb | nk<<8 | k<<16, first Vw cell (i = 0), ket block offset}
};
__global__ void __launch_bounds__(DN_WARPS * 32) k_dense3(Tables T, const uint4* __restrict__ ditems, const uint32_t* __restrict__ n_items_p,
                                                         const unsigned long long* __restrict__ recs, double* __restrict__ out)
{
    __shared__ DenseWarp3 shw[DN_WARPS];
    DenseWarp3& W = shw[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    const uint32_t n_runs = __ldg(n_items_p + 2);
    const uint32_t nt = (uint32_t)T.n_tup3;
    const double* __restrict__ dtab = T.dtab3;
    for (uint32_t it = gw; it < n_runs; it += nw) {
        const uint4 item = __ldg(ditems + it);
        const uint32_t pos0 = item.x, cnt = item.y, g = item.z, mi = item.w;
        const uint32_t tb = g / nt, tk = g - tb * nt;
        const int4 kb = __ldg(T.tk3 + tb), kk = __ldg(T.tk3 + tk);
        const uint4 sg = __ldg(T.sgrp3 + g);
        const int sjb = kb.w & 255, sjk = kk.w & 255, mm = min(sjb, sjk);
        const int imb = (int)mi + ((sjb - mm) >> 1), imk = (int)mi + ((sjk - mm) >> 1);
        const uint16_t* msb = T.mstart3 + __ldg(T.mstoff3 + tb);
        const uint16_t* msk = T.mstart3 + __ldg(T.mstoff3 + tk);
        const uint32_t s0b = __ldg(msb + imb), nmb = __ldg(msb + imb + 1) - s0b;
        const uint32_t s0k = __ldg(msk + imk), nmk = __ldg(msk + imk + 1) - s0k;
        const int Jminb = (kb.w >> 16) & 255, Jmink = (kk.w >> 16) & 255;
        const int Jlo = max(Jminb, Jmink), nblk = ((min((kb.w >> 24) & 255, (kk.w >> 24) & 255) - Jlo) >> 1) + 1;
        const int q0 = max(0, (abs(2 * imb - sjb) - Jlo + 1) >> 1);   // first J block with J >= |M|
        // flattened ket rows of the blocks q0 .. nblk-1
        int2 jb = make_int2(0, 0), jk = make_int2(0, 0);
        if (lane < nblk) {
            jb = __ldg(T.jinfo3 + kb.z + ((Jlo - Jminb) >> 1) + lane);
            jk = __ldg(T.jinfo3 + kk.z + ((Jlo - Jmink) >> 1) + lane);
        }
        const uint32_t vv = (uint32_t)(jb.y * row_pitch3(jk.y)), rk = lane >= q0 ? (uint32_t)jk.y : 0u;
        uint32_t iv = vv, ir = rk;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            uint32_t xv = __shfl_up_sync(0xFFFFFFFFu, iv, off), xr = __shfl_up_sync(0xFFFFFFFFu, ir, off);
            if (lane >= off) { iv += xv; ir += xr; }
        }
        const uint32_t R = __shfl_sync(0xFFFFFFFFu, ir, 31);   // ket rows in play (<= DENSE_RMAX by the upload's feasibility test)
        if (lane >= q0 && lane < nblk)
            for (int k = 0; k < jk.y; k++)
                W.rmap[ir - rk + k] = make_uint4((uint32_t)kb.x + (uint32_t)jb.x, (uint32_t)jb.y | ((uint32_t)jk.y << 8) | ((uint32_t)k << 16),
                                                 iv - vv + (uint32_t)k, (uint32_t)kk.x + (uint32_t)jk.x);
        // isospin bins present in the run
        uint32_t bits = 0u;
        for (uint32_t i = lane; i < cnt; i += 32) bits |= 1u << ((uint32_t)(__ldg(recs + pos0 + i) >> 24) & 31u);
        bits = __reduce_or_sync(0xFFFFFFFFu, bits);
        __syncwarp();
        const uint32_t gsize = sg.y, S = vw_stride(gsize, T.vw_f32), ldv = (nmk + 7u) & ~7u;
        const int nchunk = (int)((R + 3u) >> 2);
        const uint32_t mrow = (uint32_t)lane >> 2, kcol = (uint32_t)lane & 3u;
        for (uint32_t bin = 0; bin < (uint32_t)NBIN3; bin++) {
            if (!((bits >> bin) & 1u)) continue;   // warp-uniform
            const uint32_t* __restrict__ vwb = T.vw20 + (size_t)sg.z * 4 + (size_t)bin * S;
            for (uint32_t mt = 0; mt * 8u < nmb; mt++) {
                // A fragments: T[mu = 8 mt + lane/4][r = 4 c + lane%4] for every K chunk c
                double a[DN_CHUNKS];
                const uint32_t mu = mt * 8u + mrow;
#pragma unroll
                for (int c = 0; c < DN_CHUNKS; c++) {
                    a[c] = 0.0;
                    const uint32_t r = 4u * c + kcol;
                    if (c < nchunk && r < R && mu < nmb) {
                        const uint4 e = W.rmap[r];
                        const uint32_t nb = e.y & 255u, P = (uint32_t)row_pitch3((e.y >> 8) & 255u);
                        const double* __restrict__ cb = dtab + (e.x + (s0b + mu) * nb);
                        double t = 0.0;
                        for (uint32_t i = 0; i < nb; i++) {
                            const uint32_t cell = e.z + i * P;
                            t = fma(__ldg(cb + i), ldvw_global(vwb, gsize, cell, T.vw_f32), t);
                        }
                        a[c] = t;
                    }
                }
                for (uint32_t nt8 = 0; nt8 * 8u < nmk; nt8++) {
                    const uint32_t mup = nt8 * 8u + mrow;   // B fragment: Ck[mu' = 8 nt8 + lane/4][r = 4 c + lane%4]
                    double c0 = 0.0, c1 = 0.0;
#pragma unroll
                    for (int c = 0; c < DN_CHUNKS; c++) {
                        if (c < nchunk) {   // warp-uniform
                            const uint32_t r = 4u * c + kcol;
                            double b = 0.0;
                            if (r < R && mup < nmk) {
                                const uint4 e = W.rmap[r];
                                b = __ldg(dtab + (e.w + (s0k + mup) * ((e.y >> 8) & 255u) + (e.y >> 16)));
                            }
                            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                         : "+d"(c0), "+d"(c1) : "d"(a[c]), "d"(b));
                        }
                    }
                    *reinterpret_cast<double2*>(&W.vm[(mt * 8u + mrow) * ldv + nt8 * 8u + 2u * kcol]) = make_double2(c0, c1);
                }
            }
            __syncwarp();
            for (uint32_t i = lane; i < cnt; i += 32) {
                const unsigned long long rec = __ldg(recs + pos0 + i);
                const uint32_t lo = (uint32_t)rec;
                if (((lo >> 24) & 31u) != bin) continue;
                // a record of another tuple pair in a mis-ordered MFDN_PRESORTED stream must not index outside the buffer
                const uint32_t rb = min((lo & 0xFFFu) - s0b, nmb - 1u), rkk = min(((lo >> 12) & 0xFFFu) - s0k, nmk - 1u);
                const double v = W.vm[rb * ldv + rkk];
                out[pos0 + i] = (((lo >> 29) & 1u) ? -v : v) + 0.0;
            }
            __syncwarp();
        }
    }
}

// ------------------------------------------------------------------------------- NEXT-2: dense block mode
// Whole m-scheme blocks without a request list (PAPER.md:53-55 A' = D^T A D, Fig. 1 at :69; "at a higher level in the matrix
// construction stage").  One warp per (group, M, isospin bin): it forms
//     Vm[mu, mu'] = sum_{J >= |M|} sum_{J12, J12'} Cb[mu; J,J12] * Vw_bin[J; J12,J12'] * Ck[mu'; J,J12']
// (measured: 7.5 G entries/s on all 1415 non-empty groups of config 2, 14.8 G entries/s on 1940 groups of config 3 -- every
// warp is a chain of dependent descriptor loads for a ~10 x 10 tile, so this is latency-bound, not yet faster per entry than
// the request path)
// over ALL bra and ket m-states of that M with the same two chained products as k_dense3 (T = Cb * Vw in the A-fragment
// layout, Vm = T * Ck^T with mma.sync.m8n8k4.f64) and stores the 8 x 8 tiles straight from the accumulator fragments.
// An entry whose bra or ket is not an ordered Slater determinant (particles of one orbital not in ascending SPS order, or
// an SPS that does not exist) is stored as +0.0: its value is that of the ordered partner times the permutation sign.
struct BinPat { uint8_t v[NBIN3]; };
constexpr BinPat make_binpat()   // bin -> bra pattern << 3 | ket pattern, the enumeration of mfdn_orbitals_init
{
    BinPat p{};
    int n = 0;
    for (int tb = 0; tb < 8; tb++)
        for (int tk = 0; tk < 8; tk++) {
            int cb = (tb & 1) + ((tb >> 1) & 1) + (tb >> 2), ck = (tk & 1) + ((tk >> 1) & 1) + (tk >> 2);
            if (cb == ck) p.v[n++] = (uint8_t)(tb * 8 + tk);
        }
    return p;
}
__constant__ BinPat c_binpat = make_binpat();

struct BlockItem { uint32_t g, mi; unsigned long long off; };   // off: first entry of the (group, M) sub-block (20 bins follow each other)

// is the m-state `nat` = (ima*(jb+1)+imb)*(jc+1)+imc of a tuple with tz pattern `pat` an ordered Slater determinant?
__device__ __forceinline__ bool ordered_state3(const Tables& T, int4 orb, int4 d, uint32_t nat, int pat)
{
    const int jb1 = ((d.x >> 8) & 255) + 1, jc1 = ((d.x >> 16) & 255) + 1;
    const int imc = nat % jc1, imb = (nat / jc1) % jb1, ima = nat / (jc1 * jb1);
    const int sa = __ldg(T.spsidx3 + (orb.x * 2 + ((pat >> 2) & 1)) * 32 + ima);
    const int sb = __ldg(T.spsidx3 + (orb.y * 2 + ((pat >> 1) & 1)) * 32 + imb);
    const int sc = __ldg(T.spsidx3 + (orb.z * 2 + (pat & 1)) * 32 + imc);
    return sa >= 0 && sb >= 0 && sc >= 0 && (orb.x != orb.y || sa < sb) && (orb.y != orb.z || sb < sc);
}

__global__ void __launch_bounds__(DN_WARPS * 32) k_block3(Tables T, const BlockItem* __restrict__ items, uint32_t n_items, double* __restrict__ out)
{
    __shared__ uint4 s_rmap[DN_WARPS][DENSE_RMAX];
    uint4* rmap = s_rmap[threadIdx.x >> 5];
    const int lane = threadIdx.x & 31;
    const uint32_t gw = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, nw = (gridDim.x * blockDim.x) >> 5;
    const uint32_t nt = (uint32_t)T.n_tup3;
    const double* __restrict__ dtab = T.dtab3;
    for (uint32_t wi = gw; wi < n_items * (uint32_t)NBIN3; wi += nw) {
        const uint32_t it = wi / (uint32_t)NBIN3, bin = wi - it * (uint32_t)NBIN3;
        const BlockItem item = items[it];
        const uint32_t g = item.g, mi = item.mi;
        const uint32_t tb = g / nt, tk = g - tb * nt;
        const int4 kb = __ldg(T.tk3 + tb), kk = __ldg(T.tk3 + tk);
        const int4 db = __ldg(T.tdesc3 + tb), dk = __ldg(T.tdesc3 + tk);
        const int4 ob = __ldg(T.torb3 + tb), ok = __ldg(T.torb3 + tk);
        const uint4 sg = __ldg(T.sgrp3 + g);
        const int sjb = kb.w & 255, sjk = kk.w & 255, mm = min(sjb, sjk);
        const int imb = (int)mi + ((sjb - mm) >> 1), imk = (int)mi + ((sjk - mm) >> 1);
        const uint16_t* msb = T.mstart3 + __ldg(T.mstoff3 + tb);
        const uint16_t* msk = T.mstart3 + __ldg(T.mstoff3 + tk);
        const uint32_t s0b = __ldg(msb + imb), nmb = __ldg(msb + imb + 1) - s0b;
        const uint32_t s0k = __ldg(msk + imk), nmk = __ldg(msk + imk + 1) - s0k;
        const uint16_t* isb = T.isig3 + db.w + s0b;   // natural index of the bra / ket m-states of this M
        const uint16_t* isk = T.isig3 + dk.w + s0k;
        const int Jminb = (kb.w >> 16) & 255, Jmink = (kk.w >> 16) & 255;
        const int Jlo = max(Jminb, Jmink), nblk = ((min((kb.w >> 24) & 255, (kk.w >> 24) & 255) - Jlo) >> 1) + 1;
        const int q0 = max(0, (abs(2 * imb - sjb) - Jlo + 1) >> 1);   // first J block with J >= |M|
        int2 jb = make_int2(0, 0), jk = make_int2(0, 0);
        if (lane < nblk) {
            jb = __ldg(T.jinfo3 + kb.z + ((Jlo - Jminb) >> 1) + lane);
            jk = __ldg(T.jinfo3 + kk.z + ((Jlo - Jmink) >> 1) + lane);
        }
        const uint32_t vv = (uint32_t)(jb.y * row_pitch3(jk.y)), rk = lane >= q0 ? (uint32_t)jk.y : 0u;
        uint32_t iv = vv, ir = rk;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            uint32_t xv = __shfl_up_sync(0xFFFFFFFFu, iv, off), xr = __shfl_up_sync(0xFFFFFFFFu, ir, off);
            if (lane >= off) { iv += xv; ir += xr; }
        }
        const uint32_t R = __shfl_sync(0xFFFFFFFFu, ir, 31);   // flattened ket rows in play (<= DENSE_RMAX, checked by the host)
        __syncwarp();
        if (lane >= q0 && lane < nblk)
            for (int k = 0; k < jk.y; k++)
                rmap[ir - rk + k] = make_uint4((uint32_t)kb.x + (uint32_t)jb.x, (uint32_t)jb.y | ((uint32_t)jk.y << 8) | ((uint32_t)k << 16),
                                               iv - vv + (uint32_t)k, (uint32_t)kk.x + (uint32_t)jk.x);
        __syncwarp();
        const uint32_t gsize = sg.y, S = vw_stride(gsize, T.vw_f32);
        const int nchunk = (int)((R + 3u) >> 2);
        const uint32_t mrow = (uint32_t)lane >> 2, kcol = (uint32_t)lane & 3u;
        {
            const int patb = c_binpat.v[bin] >> 3, patk = c_binpat.v[bin] & 7;
            const uint32_t* __restrict__ vwb = T.vw20 + (size_t)sg.z * 4 + (size_t)bin * S;
            double* __restrict__ dst = out + item.off + (size_t)bin * nmb * nmk;
            for (uint32_t mt = 0; mt * 8u < nmb; mt++) {
                double a[DN_CHUNKS];
                const uint32_t mu = mt * 8u + mrow;
#pragma unroll
                for (int c = 0; c < DN_CHUNKS; c++) {
                    a[c] = 0.0;
                    const uint32_t r = 4u * c + kcol;
                    if (c < nchunk && r < R && mu < nmb) {
                        const uint4 e = rmap[r];
                        const uint32_t nb = e.y & 255u, P = (uint32_t)row_pitch3((e.y >> 8) & 255u);
                        const double* __restrict__ cb = dtab + (e.x + (s0b + mu) * nb);
                        double t = 0.0;
                        for (uint32_t i = 0; i < nb; i++) {
                            const uint32_t cell = e.z + i * P;
                            t = fma(__ldg(cb + i), ldvw_global(vwb, gsize, cell, T.vw_f32), t);
                        }
                        a[c] = t;
                    }
                }
                const bool rowok = mu < nmb && ordered_state3(T, ob, db, __ldg(isb + min(mu, nmb - 1u)), patb);
                for (uint32_t nt8 = 0; nt8 * 8u < nmk; nt8++) {
                    const uint32_t mup = nt8 * 8u + mrow;
                    double c0 = 0.0, c1 = 0.0;
#pragma unroll
                    for (int c = 0; c < DN_CHUNKS; c++) {
                        if (c < nchunk) {   // warp-uniform
                            const uint32_t r = 4u * c + kcol;
                            double b = 0.0;
                            if (r < R && mup < nmk) {
                                const uint4 e = rmap[r];
                                b = __ldg(dtab + (e.w + (s0k + mup) * ((e.y >> 8) & 255u) + (e.y >> 16)));
                            }
                            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                                         : "+d"(c0), "+d"(c1) : "d"(a[c]), "d"(b));
                        }
                    }
                    const uint32_t n0 = nt8 * 8u + 2u * kcol, n1 = n0 + 1u;
                    if (mu < nmb) {
                        if (n0 < nmk) dst[(size_t)mu * nmk + n0] = (rowok && ordered_state3(T, ok, dk, __ldg(isk + n0), patk)) ? c0 + 0.0 : 0.0;
                        if (n1 < nmk) dst[(size_t)mu * nmk + n1] = (rowok && ordered_state3(T, ok, dk, __ldg(isk + n1), patk)) ? c1 + 0.0 : 0.0;
                    }
                }
            }
        }
        __syncwarp();
    }
}

__global__ void __launch_bounds__(128) k_transform2(Tables T, long long n, const unsigned long long* __restrict__ recs,
                                                   double* __restrict__ out)
{
    const long long pos = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool valid = pos < n;
    const unsigned long long rec = valid ? __ldg(recs + pos) : ~0ull;
    const uint32_t key = (uint32_t)(rec >> REC_KEY_SHIFT);
    bool done = !valid || key == REC_INVALID;
    double result = 0.0;
    const uint32_t nt = (uint32_t)T.n_tup2;
    for (;;) {
        unsigned pending = __ballot_sync(0xFFFFFFFFu, !done);
        if (pending == 0) break;
        const uint32_t g = __shfl_sync(0xFFFFFFFFu, key, __ffs(pending) - 1);
        const bool mine = !done && key == g;
        if (mine) done = true;
        const uint32_t so = __ldg(T.slab_off2 + g);
        if (so == NO_SLAB) continue;
        const uint32_t tb = g / nt, tk = g - tb * nt;
        const int4 db = __ldg(T.tdesc2 + tb), dk = __ldg(T.tdesc2 + tk);
        const int ja = db.x & 255, jb = (db.x >> 8) & 255, jc = dk.x & 255, jd = (dk.x >> 8) & 255;
        const uint32_t mrec = mine ? (uint32_t)rec : 0u;
        const int ima = mrec & 31, imb = (mrec >> 5) & 31, imc = (mrec >> 15) & 31, imd = (mrec >> 20) & 31;
        const int tzb = mine ? (int)((rec >> 33) & 3) : 0, tzk = mine ? (int)((rec >> 30) & 3) : 0;
        const double2 w = __ldg((const double2*)T.wtab2 + (tzb * 4 + tzk));
        const int nj = T.nj;
        const int Jminb = db.y & 255, Jmink = dk.y & 255;
        const int Jlo = max(Jminb, Jmink), Jhi = min((db.y >> 8) & 255, (dk.y >> 8) & 255);
        const int Sb = (ja + 1) * (jb + 1), Sk = (jc + 1) * (jd + 1);
        const double* cb = T.cg1 + __ldg(T.cg1_off + (ja >> 1) * nj + (jb >> 1)) + ima * (jb + 1) + imb + (Jlo - Jminb) * Sb;
        const double* ck = T.cg1 + __ldg(T.cg1_off + (jc >> 1) * nj + (jd >> 1)) + imc * (jd + 1) + imd + (Jlo - Jmink) * Sk;
        const double2* cell = (const double2*)T.slab2 + so;
        double total = 0.0;
        // (a table transposed to [m-pair][J] was tried: 1.26 instead of 0.87 ms -- in this layout the lanes of a warp, whose
        // records cover the m-pairs of one group densely, read neighbouring addresses for every J)
        for (int q = 0; q <= Jhi - Jlo; q++) {
            double2 v = __ldg(cell + q);
            double c = __ldg(cb + q * Sb) * __ldg(ck + q * Sk);
            total = fma(c, fma(w.y, v.y, w.x * v.x), total);
        }
        double norm = ((db.x >> 24) & 1) ? (((dk.x >> 24) & 1) ? 2.0 : 1.4142135623730951)
                                         : (((dk.x >> 24) & 1) ? 1.4142135623730951 : 1.0);
        if (mine) result = (((rec >> 36) & 1) ? -(norm * total) : norm * total) + 0.0;
    }
    if (valid) out[pos] = result;
}

size_t align256(size_t x) { return (x + 255) & ~size_t(255); }

template <int BODY>
int run(mfdn_ctx* c, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work, size_t* work_bytes,
        uint32_t flags, void* stream, const Accum* acc = nullptr)
{
    if (!c || !work_bytes || n < 0 || n >= (int64_t)0xFFFFFFF0ll) return c ? fail(c, MFDN_ERR_ARG, "bad n / work_bytes") : MFDN_ERR_ARG;
    if (BODY == 3 ? !c->has3 : !c->has2) return fail(c, MFDN_ERR_STATE, "mscheme before coupled upload");
    if ((flags & MFDN_FORCE_DENSE) && (BODY != 3 || (flags & MFDN_FORCE_NAIVE)))
        return fail(c, MFDN_ERR_ARG, "MFDN_FORCE_DENSE: 3-body only, not together with MFDN_FORCE_NAIVE");
    const int u16 = (flags & MFDN_REQ_U16) ? 1 : 0;
    if (u16 && c->t.n_sps > 65536) return fail(c, MFDN_ERR_ARG, "MFDN_REQ_U16 needs at most 65536 single-particle states");
    const long long nt = BODY == 3 ? c->t.n_tup3 : c->t.n_tup2;
    if (nt * nt >= (long long)REC_INVALID) return fail(c, MFDN_ERR_ARG, "too many tuples for 27-bit group keys");
    // sort buckets: 2-body one per group, 3-body one per (group, M); last bucket: requests failing S1-S6
    const long long n_buckets = (BODY == 3 ? (long long)c->t.n_buckets3 : nt * nt) + 1;
    const long long n_tiles = (n_buckets + SCAN_TILE - 1) / SCAN_TILE;
    // Path choice by batch size.  The paths give the same values bit for bit (same operations in the same order), so the choice
    // is invisible in the results.  Thread-per-request needs no sort and no per-table scans, whose cost is fixed per call
    // (config 3: ~150 us at any n).  Measured cross-overs on B200: 2-body: thread per request at every n up
    // to 2^26 (~6 terms per request: sorting costs more than it saves; 2.69 against 3.08 ms at 2^26); 3-body: k_direct3 up to
    // 2^20 requests (config 3: 45 against 124 us at 2^14, 304 against 379 us at 2^20), then the one-pass scatter / gather up to
    // 2^23 requests, the two-pass partition above.  Any flag that names a path overrides the choice.
    // MFDN_PRESORTED is a property of the input, not a path: a pre-sorted 2-body batch is still fastest thread-per-request
    // (1.03 against 1.30 ms at 2^26), and so is a small pre-sorted 3-body batch.
    const bool named = flags & (MFDN_FORCE_DENSE | MFDN_ONE_PASS_SORT | MFDN_FORCE_SORT);
    const bool auto_direct = !named && (BODY == 2 || n <= (c->vw_bytes3 <= (64ll << 20) ? 2 * MFDN_DIRECT3_MAX : MFDN_DIRECT3_MAX));
    const bool naive = (flags & MFDN_FORCE_NAIVE) || auto_direct;
    const bool sort = !naive && !(flags & MFDN_PRESORTED);
    const bool items = !naive && BODY == 3;    // the 3-body transform walks a list of one-group work items
    const bool hist_needed = sort || items;
    // work items: at most 5 rounds per chunk of a group with more than SMALL_ITEM3 records; one entry per small group
    // or per SMALL_ITEM3 records of an oversized one
    const long long max_items = 5 * (n / ITEM3 + n / (SMALL_ITEM3 + 1) + 1) + n / SMALL_ITEM3 + std::min<long long>(n, nt * nt + 1) + 1;
    size_t need = 256;
    const bool dense = items && (flags & MFDN_FORCE_DENSE);
    const long long max_ditems = dense ? std::min<long long>(n, n_buckets) + 1 : 0;
    // sort path: coarse bins of the two-pass partition = bucket >> csh with about as many bins as buckets per bin
    int csh = 0;
    while ((1ll << (2 * csh)) < n_buckets) csh++;
    csh = std::min(csh, 12);   // PART_NF = 4096 buckets per bin at most
    while (((n_buckets + (1ll << csh) - 1) >> csh) > PART_NC) csh++;
    const bool two_pass = sort && csh <= 12 && !(flags & MFDN_ONE_PASS_SORT) && ((flags & MFDN_FORCE_SORT) || n >= MFDN_TWO_PASS_MIN);
    const int nc = (int)((n_buckets + (1ll << csh) - 1) >> csh);
    const long long n_ktiles = (n + KEYS_PER_BLOCK - 1) / KEYS_PER_BLOCK, n_chunks = (n_ktiles + TS_CHUNK - 1) / TS_CHUNK;
    const long long max_tiles2 = n_ktiles + nc;
    size_t o_recs = 0, o_p1rec = 0, o_map1 = 0, o_map2 = 0, o_slot1 = 0, o_slot2 = 0, o_tcnt = 0, o_part = 0, o_cstart = 0, o_tiles2 = 0,
           o_hist = 0, o_sums = 0, o_items = 0, o_count = 0, o_ditems = 0;
    if (!naive) {
        need = o_recs + align256((size_t)n * 8);
        if (sort) {
            o_p1rec = need;
            o_map1 = o_p1rec + align256((size_t)n * 8);
            need = o_map1 + align256((size_t)n * 4);
        }
        if (two_pass) {
            o_map2 = need;
            o_slot1 = o_map2 + align256((size_t)n * 4);
            o_slot2 = o_slot1 + align256((size_t)n * 2);
            o_tcnt = o_slot2 + align256((size_t)n * 2);
            o_part = o_tcnt + align256((size_t)n_ktiles * nc * 4);
            o_cstart = o_part + align256((size_t)n_chunks * nc * 4);
            o_tiles2 = o_cstart + align256((size_t)(nc + 1) * 4);
            need = o_tiles2 + align256((size_t)(max_tiles2 + 1) * 16);
        }
        if (hist_needed) {
            o_hist = need;
            o_sums = o_hist + align256((size_t)n_buckets * 4);
            need = o_sums + align256((size_t)n_tiles * 4);
        }
        if (items) {
            o_items = need;
            o_count = o_items + align256((size_t)max_items * 16);
            o_ditems = o_count + 256;
            need = o_ditems + align256((size_t)max_ditems * 16);
        }
    }
    // NEXT-1: on every path but the default one the values go to scratch in request order and are accumulated from there
    const bool acc_fused = acc && two_pass;
    size_t o_accvals = 0;
    if (acc && !acc_fused) {
        o_accvals = align256(need);
        need = o_accvals + align256((size_t)n * 8);
    }
    if (!d_work) { *work_bytes = need; return MFDN_OK; }
    if (*work_bytes < need) return fail(c, MFDN_ERR_OOM, "scratch too small");
    if (n == 0) return MFDN_OK;
    if (acc) {
        if (!acc->loc || !acc->H || acc->h_len < 0) return fail(c, MFDN_ERR_ARG, "null location / target pointer");
        d_out = acc_fused ? nullptr : (double*)((char*)d_work + o_accvals);
    }
    if (!d_req || (!d_out && !acc)) return fail(c, MFDN_ERR_ARG, "null request/output pointer");
    cudaStream_t st = (cudaStream_t)stream;
    mfdn_ctx::EvTriple ev{nullptr, nullptr, nullptr, nullptr, sort};
    MFDN_CUDA(c, cudaSetDevice(c->device));   // the tables live on the context's device, whatever the caller's current one
    if (c->profile) {
        cudaEvent_t* e3[4] = {&ev.a, &ev.b, &ev.d, &ev.c};
        for (auto pe : e3) {
            {
                std::lock_guard<std::mutex> lk(c->mu);
                if (!c->ev_pool.empty()) { *pe = c->ev_pool.back(); c->ev_pool.pop_back(); continue; }
            }
            MFDN_CUDA(c, cudaEventCreate(pe));
        }
        MFDN_CUDA(c, cudaEventRecord(ev.a, st));
    }
    if (naive) {
        if (c->profile) MFDN_CUDA(c, cudaEventRecord(ev.b, st));
        if (BODY == 3 && !(flags & MFDN_FORCE_NAIVE)) k_direct3<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(c->t, n, d_req, d_out, d_mask, u16);
        else k_mscheme_naive<BODY><<<(unsigned)((n + 127) / 128), 128, 0, st>>>(c->t, n, d_req, d_out, d_mask, u16);
        c->launches += 1;
        if (c->profile) MFDN_CUDA(c, cudaEventRecord(ev.d, st));
    } else {
        char* w = (char*)d_work;
        unsigned long long* recs = (unsigned long long*)(w + o_recs);
        const unsigned long long* trecs = recs;
        uint32_t* hist = hist_needed ? (uint32_t*)(w + o_hist) : nullptr;
        uint32_t* sums = hist_needed ? (uint32_t*)(w + o_sums) : nullptr;
        const uint32_t invalid_bucket = (uint32_t)(n_buckets - 1);
        if (hist_needed) MFDN_CUDA(c, cudaMemsetAsync(hist, 0, (size_t)n_buckets * 4, st));
        const bool sm = c->t.n_sps <= KEYS_SPS_SMEM && (BODY == 2 || (c->t.ab3 && c->t.n_orb * c->t.n_orb <= KEYS_AB_SMEM));
        const unsigned gkb = (unsigned)((n + KEYS_PER_BLOCK - 1) / KEYS_PER_BLOCK);
        // 3-body with every per-basis table in shared memory (k_keys3s) when they fit; MFDN_ONE_PASS_SORT keeps the general kernel
        KeysSmem3 L{};
        bool smem_keys = false, late_hist = false;
        if (BODY == 3 && sm && c->t.ncls3 > 0 && !(flags & MFDN_ONE_PASS_SORT)) {
            auto up = [](uint32_t x) { return (x + 15u) & ~15u; };
            L.tdesc = 0;
            L.stm = up(L.tdesc + (uint32_t)nt * 16u);
            L.ab = up(L.stm + (uint32_t)c->t.stm12_len3 * 8u);
            L.sps = up(L.ab + (uint32_t)(c->t.n_orb * c->t.n_orb) * 8u);
            L.rowbase = up(L.sps + (uint32_t)c->t.n_sps * 4u);
            L.ch = up(L.rowbase + (uint32_t)nt * 4u);
            L.colcum = up(L.ch + 2u * (uint32_t)PART_NC * 4u);
            L.sig = up(L.colcum + (uint32_t)(c->t.ncls3 * nt) * 2u);
            L.tzbin = up(L.sig + (uint32_t)c->t.sig_len3 * 2u);
            L.total = L.tzbin + 64u;
            smem_keys = L.total <= 200u * 1024u;
        }
        if (smem_keys) {
            if (!c->keys_attr_set.load()) {   // benign if two threads do it at once
                MFDN_CUDA(c, (cudaFuncSetAttribute(k_keys3s<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)));
                MFDN_CUDA(c, (cudaFuncSetAttribute(k_keys3s<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)));
                MFDN_CUDA(c, (cudaFuncSetAttribute(k_keys3s<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)));
                MFDN_CUDA(c, (cudaFuncSetAttribute(k_keys3s<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024)));
                c->keys_attr_set.store(true);
            }
            const unsigned gks = (unsigned)std::min<long long>(n_ktiles, c->num_sms);
            uint32_t* tc = sort && two_pass ? (uint32_t*)(w + o_tcnt) : nullptr;
            late_hist = sort && two_pass;   // the buckets are then counted by k_count2 after pass 1
            const int tsh = sort ? csh : 0, tnc = sort ? nc : 0;
            auto kern = sort ? (u16 ? k_keys3s<false, true> : k_keys3s<false, false>) : (u16 ? k_keys3s<true, true> : k_keys3s<true, false>);
            kern<<<gks, KS_THREADS, L.total, st>>>(c->t, L, n, d_req, recs, d_mask, late_hist ? nullptr : hist, invalid_bucket, tc, tsh, tnc, (int)n_ktiles);
        } else if (sort) {
            uint32_t* tcnt = two_pass ? (uint32_t*)(w + o_tcnt) : nullptr;
            if (sm) k_keys<BODY, false, true><<<gkb, 256, 0, st>>>(c->t, n, d_req, recs, d_mask, hist, invalid_bucket, nullptr, tcnt, csh, nc, u16);
            else k_keys<BODY, false, false><<<gkb, 256, 0, st>>>(c->t, n, d_req, recs, d_mask, hist, invalid_bucket, nullptr, tcnt, csh, nc, u16);
        } else {
            if (sm) k_keys<BODY, true, true><<<gkb, 256, 0, st>>>(c->t, n, d_req, recs, d_mask, hist, invalid_bucket, nullptr, nullptr, 0, 0, u16);
            else k_keys<BODY, true, false><<<gkb, 256, 0, st>>>(c->t, n, d_req, recs, d_mask, hist, invalid_bucket, nullptr, nullptr, 0, 0, u16);
        }
        c->launches += 1;
        if (hist_needed && !late_hist) {
            k_scan_tiles<<<(unsigned)n_tiles, SCAN_T, 0, st>>>(hist, n_buckets, sums);
            k_scan_sums<<<1, 1024, 0, st>>>(sums, (int)n_tiles);
            k_scan_add<<<(unsigned)n_tiles, SCAN_T, 0, st>>>(hist, n_buckets, sums);
            c->launches += 3;
        }
        double* tout = d_out;   // where the transform writes: request order if pre-sorted, else bucket order (scratch)
        unsigned long long* p1rec = (unsigned long long*)(w + o_p1rec);
        uint32_t *map1 = (uint32_t*)(w + o_map1), *map2 = (uint32_t*)(w + o_map2);
        uint16_t *slot1 = (uint16_t*)(w + o_slot1), *slot2 = (uint16_t*)(w + o_slot2);
        uint4* tiles2 = (uint4*)(w + o_tiles2);
        if (two_pass) {
            uint32_t* tcnt = (uint32_t*)(w + o_tcnt);
            uint32_t* part = (uint32_t*)(w + o_part);
            uint32_t* cstart = (uint32_t*)(w + o_cstart);
            if (!c->part_attr_set.load()) {   // benign if two threads do it at once
                MFDN_CUDA(c, cudaFuncSetAttribute(k_part<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, PART_SMEM));
                MFDN_CUDA(c, cudaFuncSetAttribute(k_part<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, PART_SMEM));
                MFDN_CUDA(c, cudaFuncSetAttribute(k_back<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, KEYS_PER_BLOCK * 8));
                MFDN_CUDA(c, cudaFuncSetAttribute(k_back<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, KEYS_PER_BLOCK * 8));
                MFDN_CUDA(c, (cudaFuncSetAttribute(k_back<1, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, KEYS_PER_BLOCK * 8)));
                c->part_attr_set.store(true);
            }
            const dim3 gts((unsigned)((nc + 127) / 128), (unsigned)n_chunks);
            k_tscan_sum<<<gts, 128, 0, st>>>(tcnt, (int)n_ktiles, nc, part);
            k_tscan_mid<<<1, 1024, 0, st>>>(part, (int)n_chunks, nc, cstart);
            k_tscan_fill<<<gts, 128, 0, st>>>(tcnt, (int)n_ktiles, nc, part, cstart);
            k_tiles2<<<1, 1024, 0, st>>>(cstart, nc, tiles2);
            k_part<1><<<gkb, P_THREADS, PART_SMEM, st>>>(n, recs, tcnt, nullptr, nullptr, csh, nc, p1rec, map1, slot1, invalid_bucket);
            if (late_hist) {
                k_count2<<<(unsigned)max_tiles2, P_THREADS, 0, st>>>(p1rec, tiles2, hist, csh, invalid_bucket);
                k_scan_tiles<<<(unsigned)n_tiles, SCAN_T, 0, st>>>(hist, n_buckets, sums);
                k_scan_sums<<<1, 1024, 0, st>>>(sums, (int)n_tiles);
                k_scan_add<<<(unsigned)n_tiles, SCAN_T, 0, st>>>(hist, n_buckets, sums);
                c->launches += 4;
            }
            // the request-order records are dead after pass 1: the bucket-ordered records take their place
            k_part<2><<<(unsigned)max_tiles2, P_THREADS, PART_SMEM, st>>>(n, p1rec, nullptr, tiles2, hist, csh, 1 << csh, recs, map2, slot2, invalid_bucket);
            c->launches += 6;
            tout = (double*)p1rec;   // ... and the coarse-ordered records are dead after pass 2: the values take theirs
        } else if (sort) {
            k_scatter<<<(unsigned)((n + 256 * SC_PER_THREAD - 1) / (256 * SC_PER_THREAD)), 256, 0, st>>>(n, recs, hist, p1rec, map1, invalid_bucket);
            c->launches += 1;
            trecs = p1rec;
            tout = (double*)recs;   // the request-order records are dead after the scatter: reuse them for the values
        }
        if (items) {
            uint4* itm = (uint4*)(w + o_items);
            uint32_t* cnt = (uint32_t*)(w + o_count);
            MFDN_CUDA(c, cudaMemsetAsync(cnt, 0, 16, st));
            uint4* ditm = (uint4*)(w + o_ditems);
            const uint32_t last_slot = (uint32_t)(max_items - 1);
            k_items3<<<(unsigned)((nt * nt + 1 + 255) / 256), 256, 0, st>>>(hist, c->t.gbase3, (uint32_t)(nt * nt), (uint32_t)n_buckets, sort ? 1 : 0,
                                                                             (uint32_t)n, c->t.sgrp3, itm, last_slot, cnt, dense ? 0.f : -1.f, ditm, c->t.vw_f32);
            if (c->profile) MFDN_CUDA(c, cudaEventRecord(ev.b, st));
            int per_sm = c->tr_blocks_per_sm.load();
            if (per_sm == 0) {   // benign if two threads do it at once: both store the same number
                MFDN_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_transform3<false>, TR_THREADS, 0));
                per_sm = std::max(per_sm, 1);
                c->tr_blocks_per_sm.store(per_sm);
            }
            const unsigned grid = (unsigned)std::min<long long>(max_items, (long long)c->num_sms * per_sm);
            if (c->t.vw_f32) k_transform3<true><<<grid, TR_THREADS, 0, st>>>(c->t, itm, cnt, trecs, tout, cnt + 3);
            else k_transform3<false><<<grid, TR_THREADS, 0, st>>>(c->t, itm, cnt, trecs, tout, cnt + 3);
            const unsigned grid_s = (unsigned)std::min<long long>((std::min<long long>(n, nt * nt + 1) + 3) / 4, (long long)c->num_sms * 16);
            if (c->t.vw_f32) k_transform3_small<true><<<grid_s, 128, 0, st>>>(c->t, itm, last_slot, cnt, trecs, tout);
            else k_transform3_small<false><<<grid_s, 128, 0, st>>>(c->t, itm, last_slot, cnt, trecs, tout);
            c->launches += 3;
            if (dense) {
                const unsigned grid_d = (unsigned)std::min<long long>((max_ditems + DN_WARPS - 1) / DN_WARPS, (long long)c->num_sms * 8);
                k_dense3<<<grid_d, DN_WARPS * 32, 0, st>>>(c->t, ditm, cnt, trecs, tout);
                c->launches += 1;
            }
        } else {
            if (c->profile) MFDN_CUDA(c, cudaEventRecord(ev.b, st));
            k_transform2<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(c->t, n, trecs, tout);
            c->launches += 1;
        }
        if (c->profile) MFDN_CUDA(c, cudaEventRecord(ev.d, st));
        if (two_pass) {
            double* tmp = (double*)recs;   // the bucket-ordered records are dead after the transform
            k_back<2><<<(unsigned)max_tiles2, P_THREADS, KEYS_PER_BLOCK * 8, st>>>(n, tout, tiles2, map2, slot2, tmp, Accum{});
            if (acc) k_back<1, true><<<gkb, P_THREADS, KEYS_PER_BLOCK * 8, st>>>(n, tmp, nullptr, map1, slot1, nullptr, *acc);
            else k_back<1><<<gkb, P_THREADS, KEYS_PER_BLOCK * 8, st>>>(n, tmp, nullptr, map1, slot1, d_out, Accum{});
            c->launches += 2;
        } else if (sort) {
            k_unpermute<<<(unsigned)((n + 256 * SC_PER_THREAD - 1) / (256 * SC_PER_THREAD)), 256, 0, st>>>(n, tout, map1, d_out);
            c->launches += 1;
        }
    }
    if (acc && !acc_fused) {
        k_accumulate<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, d_out, *acc);
        c->launches += 1;
    }
    MFDN_CUDA(c, cudaGetLastError());
    if (c->profile) {
        MFDN_CUDA(c, cudaEventRecord(ev.c, st));
        std::lock_guard<std::mutex> lk(c->mu);
        c->ev_pending.push_back(ev);
    }
    return MFDN_OK;
}

// register-resident DFMA chains: 8 independent accumulators per thread, no memory traffic
__global__ void __launch_bounds__(256) k_fp64_peak(double* out, int iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; i++) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    double s = x0 + x1 + x2 + x3 + x4 + x5 + x6 + x7;
    if (s == 12345.678) out[0] = s;   // never true; keeps the chains alive
}

}  // namespace

extern "C" int mfdn_mscheme_2b(mfdn_ctx* c, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work,
                               size_t* work_bytes, uint32_t flags, void* stream)
{
    return run<2>(c, n, d_req, d_out, d_mask, d_work, work_bytes, flags, stream);
}

extern "C" int mfdn_mscheme_3b(mfdn_ctx* c, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, void* d_work,
                               size_t* work_bytes, uint32_t flags, void* stream)
{
    return run<3>(c, n, d_req, d_out, d_mask, d_work, work_bytes, flags, stream);
}

// ------------------------------------------------------------------------------- allocation-free call
// mfdn_mscheme_static: run<BODY>() with its scratch in an array that is part of the library image (include/mfdn_b200.h).
// In host code `g_static_scratch` is the host-side stand-in of the symbol, NOT a device address: the kernels are given the
// address cudaGetSymbolAddress returns, looked up once per device with that device current and kept in g_static_ptr.
// Every call on a device shares the array and finds the previous call's contents in it; run() never assumes zeroed
// scratch (it clears the histogram and the work-item counters on the call's stream), so nothing else needs clearing.
static __device__ __align__(256) unsigned char g_static_scratch[MFDN_STATIC_SCRATCH_BYTES];
static std::mutex g_static_mu;
constexpr int STATIC_MAX_DEVICES = 64;
static void* g_static_ptr[STATIC_MAX_DEVICES] = {};

extern "C" int mfdn_mscheme_static(mfdn_ctx* c, int body, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, uint32_t flags,
                                   void* stream)
{
    if (!c) return MFDN_ERR_ARG;
    if (body != 2 && body != 3) return fail(c, MFDN_ERR_ARG, "body must be 2 or 3");
    if (n < 0) return fail(c, MFDN_ERR_ARG, "negative request count");
    if (c->profile) return fail(c, MFDN_ERR_STATE, "mfdn_mscheme_static: not while mfdn_profile is on (profiling creates events)");
    if (c->device < 0 || c->device >= STATIC_MAX_DEVICES) return fail(c, MFDN_ERR_ARG, "mfdn_mscheme_static: device ordinal above 63");
    void* scratch = nullptr;
    {
        std::lock_guard<std::mutex> lk(g_static_mu);
        scratch = g_static_ptr[c->device];
        if (!scratch) {   // set-up, once per device
            MFDN_CUDA(c, cudaSetDevice(c->device));
            MFDN_CUDA(c, cudaGetSymbolAddress(&scratch, g_static_scratch));
            if (!scratch) return fail(c, MFDN_ERR_CUDA, "cudaGetSymbolAddress returned a null address");
            g_static_ptr[c->device] = scratch;
        }
    }
    // what this (n, flags) needs: the query form of the ordinary call (host arithmetic only)
    size_t need = 0;
    int rc = body == 3 ? run<3>(c, n, nullptr, nullptr, nullptr, nullptr, &need, flags, nullptr)
                       : run<2>(c, n, nullptr, nullptr, nullptr, nullptr, &need, flags, nullptr);
    if (rc != MFDN_OK) return rc;
    if (need > (size_t)MFDN_STATIC_SCRATCH_BYTES) {
        char msg[192];
        snprintf(msg, sizeof msg, "mfdn_mscheme_static: %lld requests need %zu bytes of scratch, the static array holds %zu: split the batch or use mfdn_mscheme_%db",
                 (long long)n, need, (size_t)MFDN_STATIC_SCRATCH_BYTES, body);
        return fail(c, MFDN_ERR_OOM, msg);
    }
    if (n == 0) return MFDN_OK;
    size_t have = (size_t)MFDN_STATIC_SCRATCH_BYTES;
    return body == 3 ? run<3>(c, n, d_req, d_out, d_mask, scratch, &have, flags, stream)
                     : run<2>(c, n, d_req, d_out, d_mask, scratch, &have, flags, stream);
}

extern "C" int mfdn_mscheme_accumulate_2b(mfdn_ctx* c, int64_t n, const int32_t* d_req, const int64_t* d_loc, const double* d_phase,
                                          double* d_H, int64_t h_len, uint8_t* d_mask, void* d_work, size_t* work_bytes, uint32_t flags,
                                          void* stream)
{
    const Accum a{(const long long*)d_loc, d_phase, d_H, (long long)h_len};
    return run<2>(c, n, d_req, nullptr, d_mask, d_work, work_bytes, flags, stream, &a);
}

extern "C" int mfdn_mscheme_accumulate_3b(mfdn_ctx* c, int64_t n, const int32_t* d_req, const int64_t* d_loc, const double* d_phase,
                                          double* d_H, int64_t h_len, uint8_t* d_mask, void* d_work, size_t* work_bytes, uint32_t flags,
                                          void* stream)
{
    const Accum a{(const long long*)d_loc, d_phase, d_H, (long long)h_len};
    return run<3>(c, n, d_req, nullptr, d_mask, d_work, work_bytes, flags, stream, &a);
}

// ---- NEXT-2 host side: which (M, bin) sub-blocks a group has and how long they are
namespace {
struct GroupShape {
    int tb = -1, tk = -1;
    bool empty = true;       // tuple not listed, other parity, or no common J: the block has no entries
    int mm = 0, sjb = 0, sjk = 0;
    int rows = 0;            // flattened ket rows (J, J12'), all J of the group
};
int group_shape3(mfdn_ctx* c, const int32_t* o, GroupShape& G)
{
    const int No = c->t.n_orb;
    for (int k = 0; k < 6; k++)
        if (o[k] < 0 || o[k] >= No) return fail(c, MFDN_ERR_ARG, "orbital index out of range");
    if (o[0] > o[1] || o[1] > o[2] || o[3] > o[4] || o[4] > o[5]) return fail(c, MFDN_ERR_ARG, "orbitals of a block must be ascending (a <= b <= c)");
    G.tb = c->h_tuple_id3[((size_t)o[0] * No + o[1]) * No + o[2]];
    G.tk = c->h_tuple_id3[((size_t)o[3] * No + o[4]) * No + o[5]];
    if (G.tb < 0 || G.tk < 0) return MFDN_OK;
    const uint4 sg = c->h_sgrp3[(size_t)G.tb * c->t.n_tup3 + G.tk];
    if (sg.x == NO_SLAB) return MFDN_OK;
    const int4 db = c->h_tdesc3[G.tb], dk = c->h_tdesc3[G.tk];
    G.sjb = (db.x & 255) + ((db.x >> 8) & 255) + ((db.x >> 16) & 255);
    G.sjk = (dk.x & 255) + ((dk.x >> 8) & 255) + ((dk.x >> 16) & 255);
    G.mm = std::min(G.sjb, G.sjk);
    const int Jlo = std::max((db.y >> 16) & 255, (dk.y >> 16) & 255), Jhi = std::min((db.y >> 24) & 255, (dk.y >> 24) & 255);
    const int jf = (dk.x >> 16) & 255;
    for (int twoJ = Jlo; twoJ <= Jhi; twoJ += 2) {
        const int lo = std::max(dk.y & 255, std::abs(twoJ - jf) >> 1), hi = std::min((dk.y >> 8) & 255, (twoJ + jf) >> 1);
        G.rows += std::max(0, hi - lo + 1);
    }
    G.empty = false;
    return MFDN_OK;
}
// m-states of the bra and of the ket at the mi-th common M
void m_counts3(const mfdn_ctx* c, const GroupShape& G, int mi, int64_t& nmb, int64_t& nmk)
{
    const uint16_t* msb = c->h_mstart3.data() + c->h_mstoff3[G.tb];
    const uint16_t* msk = c->h_mstart3.data() + c->h_mstoff3[G.tk];
    const int ib = mi + (G.sjb - G.mm) / 2, ik = mi + (G.sjk - G.mm) / 2;
    nmb = msb[ib + 1] - msb[ib];
    nmk = msk[ik + 1] - msk[ik];
}
}  // namespace

extern "C" int mfdn_mscheme_block_len_3b(mfdn_ctx* c, const int32_t* orbitals, int64_t* n_values)
{
    if (!c || !orbitals || !n_values) return c ? fail(c, MFDN_ERR_ARG, "null argument") : MFDN_ERR_ARG;
    if (!c->has3) return fail(c, MFDN_ERR_STATE, "block_len before coupled upload");
    GroupShape G;
    int rc = group_shape3(c, orbitals, G);
    if (rc) return rc;
    int64_t total = 0;
    if (!G.empty)
        for (int mi = 0; mi <= G.mm; mi++) {
            int64_t nmb, nmk;
            m_counts3(c, G, mi, nmb, nmk);
            total += (int64_t)NBIN3 * nmb * nmk;
        }
    *n_values = total;
    return MFDN_OK;
}

extern "C" int mfdn_mscheme_blocks_3b(mfdn_ctx* c, int64_t n_groups, const int32_t* h_orbitals, const int64_t* h_off, double* d_out,
                                      void* d_work, size_t* work_bytes, void* stream)
{
    if (!c || !work_bytes || n_groups < 0 || (n_groups > 0 && !h_orbitals)) return c ? fail(c, MFDN_ERR_ARG, "bad argument") : MFDN_ERR_ARG;
    if (!c->has3) return fail(c, MFDN_ERR_STATE, "blocks before coupled upload");
    std::vector<BlockItem> items;
    for (int64_t k = 0; k < n_groups; k++) {
        GroupShape G;
        int rc = group_shape3(c, h_orbitals + 6 * k, G);
        if (rc) return rc;
        if (G.empty) continue;
        if (G.rows > DENSE_RMAX) return fail(c, MFDN_ERR_ARG, "block mode: group with more than 64 (J, J12') ket rows");
        unsigned long long off = d_work && h_off ? (unsigned long long)h_off[k] : 0ull;
        for (int mi = 0; mi <= G.mm; mi++) {
            int64_t nmb, nmk;
            m_counts3(c, G, mi, nmb, nmk);
            if (nmb > 0 && nmk > 0) items.push_back(BlockItem{(uint32_t)((size_t)G.tb * c->t.n_tup3 + G.tk), (uint32_t)mi, off});
            off += (unsigned long long)NBIN3 * nmb * nmk;
        }
    }
    const size_t need = std::max<size_t>(256, items.size() * sizeof(BlockItem));
    if (!d_work) { *work_bytes = need; return MFDN_OK; }
    if (*work_bytes < need) return fail(c, MFDN_ERR_OOM, "scratch too small");
    if (items.empty()) return MFDN_OK;
    if (!d_out || !h_off) return fail(c, MFDN_ERR_ARG, "null output / offset pointer");
    if (items.size() >= 0xFFFFFFF0ull / NBIN3) return fail(c, MFDN_ERR_ARG, "too many (group, M) sub-blocks in one call");
    cudaStream_t st = (cudaStream_t)stream;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    // pageable source: the copy is staged before cudaMemcpyAsync returns, `items` may go out of scope
    MFDN_CUDA(c, cudaMemcpyAsync(d_work, items.data(), items.size() * sizeof(BlockItem), cudaMemcpyHostToDevice, st));
    const unsigned grid = (unsigned)std::min<size_t>((items.size() * NBIN3 + DN_WARPS - 1) / DN_WARPS, (size_t)c->num_sms * 8);
    k_block3<<<grid, DN_WARPS * 32, 0, st>>>(c->t, (const BlockItem*)d_work, (uint32_t)items.size(), d_out);
    c->launches += 1;
    MFDN_CUDA(c, cudaGetLastError());
    return MFDN_OK;
}

extern "C" int mfdn_group_keys(mfdn_ctx* c, int body, int64_t n, const int32_t* d_req, uint32_t* d_key, void* stream)
{
    if (!c || (body != 2 && body != 3) || n < 0 || !d_key || (n > 0 && !d_req)) return c ? fail(c, MFDN_ERR_ARG, "bad argument") : MFDN_ERR_ARG;
    if (body == 3 ? !c->has3 : !c->has2) return fail(c, MFDN_ERR_STATE, "group_keys before coupled upload");
    if (n == 0) return MFDN_OK;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    cudaStream_t st = (cudaStream_t)stream;
    if (body == 3) k_keys<3, false, false><<<(unsigned)((n + KEYS_PER_BLOCK - 1) / KEYS_PER_BLOCK), 256, 0, st>>>(c->t, n, d_req, nullptr, nullptr, nullptr, 0u, d_key, nullptr, 0, 0, 0);
    else k_keys<2, false, false><<<(unsigned)((n + KEYS_PER_BLOCK - 1) / KEYS_PER_BLOCK), 256, 0, st>>>(c->t, n, d_req, nullptr, nullptr, nullptr, 0u, d_key, nullptr, 0, 0, 0);
    MFDN_CUDA(c, cudaGetLastError());
    return MFDN_OK;
}

extern "C" int mfdn_profile(mfdn_ctx* c, int enable)
{
    if (!c) return MFDN_ERR_ARG;
    c->profile = enable != 0;
    return MFDN_OK;
}

extern "C" int mfdn_profile_read(mfdn_ctx* c, double* ms_sort, double* ms_transform, double* ms_unpermute, int64_t* calls)
{
    if (!c || !ms_sort || !ms_transform || !ms_unpermute || !calls) return MFDN_ERR_ARG;
    *ms_sort = *ms_transform = *ms_unpermute = 0.0;
    *calls = 0;
    std::vector<mfdn_ctx::EvTriple> pending;
    {
        std::lock_guard<std::mutex> lk(c->mu);
        pending.swap(c->ev_pending);
    }
    for (auto& ev : pending) {
        MFDN_CUDA(c, cudaEventSynchronize(ev.c));
        float t1 = 0.f, t2 = 0.f, t3 = 0.f;
        MFDN_CUDA(c, cudaEventElapsedTime(&t1, ev.a, ev.b));
        MFDN_CUDA(c, cudaEventElapsedTime(&t2, ev.b, ev.d));
        MFDN_CUDA(c, cudaEventElapsedTime(&t3, ev.d, ev.c));
        *ms_sort += t1;
        *ms_transform += t2;
        *ms_unpermute += t3;
        *calls += 1;
        std::lock_guard<std::mutex> lk(c->mu);
        c->ev_pool.push_back(ev.a); c->ev_pool.push_back(ev.b); c->ev_pool.push_back(ev.d); c->ev_pool.push_back(ev.c);
    }
    return MFDN_OK;
}

extern "C" int mfdn_fp64_peak(mfdn_ctx* c, double* tflops)
{
    if (!c || !tflops) return MFDN_ERR_ARG;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    cudaEvent_t a, b;
    MFDN_CUDA(c, cudaEventCreate(&a));
    MFDN_CUDA(c, cudaEventCreate(&b));
    const int iters = 1 << 14, blocks = c->num_sms * 8, threads = 256;
    double best = 0.0;
    for (int rep = 0; rep < 5; rep++) {
        MFDN_CUDA(c, cudaEventRecord(a, 0));
        k_fp64_peak<<<blocks, threads>>>((double*)c->t.bad_count + 8, iters, 0.999999, 1e-9);
        MFDN_CUDA(c, cudaEventRecord(b, 0));
        MFDN_CUDA(c, cudaEventSynchronize(b));
        float ms = 0.f;
        MFDN_CUDA(c, cudaEventElapsedTime(&ms, a, b));
        double tf = 2.0 * 8.0 * iters * (double)blocks * threads / (ms * 1e-3) * 1e-12;
        if (rep > 0 && tf > best) best = tf;
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    *tflops = best;
    return MFDN_OK;
}

// Measurement hook for multi-client operation: n_threads host threads, each with its own stream and its own
// scratch, push the device-resident requests through the context in chunks (thread t takes chunks t, t + n_threads, ...);
// *seconds = wall clock from the first launch to the last result.  What a many-threaded MFDn rank would do, without the
// interpreter in the way.
extern "C" int mfdn_multi_client(mfdn_ctx* c, int body, int64_t n, const int32_t* d_req, double* d_out, uint8_t* d_mask, int64_t chunk,
                                 int n_threads, uint32_t flags, double* seconds)
{
    if (!c || (body != 2 && body != 3) || n < 0 || chunk <= 0 || n_threads <= 0 || n_threads > 64 || !seconds || !d_req || !d_out)
        return c ? fail(c, MFDN_ERR_ARG, "bad argument") : MFDN_ERR_ARG;
    size_t wb = 0;
    int rc = body == 3 ? run<3>(c, chunk, nullptr, nullptr, nullptr, nullptr, &wb, flags, nullptr)
                       : run<2>(c, chunk, nullptr, nullptr, nullptr, nullptr, &wb, flags, nullptr);
    if (rc) return rc;
    MFDN_CUDA(c, cudaSetDevice(c->device));
    std::vector<cudaStream_t> st(n_threads, nullptr);
    std::vector<void*> work(n_threads, nullptr);
    std::vector<int> status(n_threads, MFDN_OK);
    cudaError_t e = cudaSuccess;
    for (int t = 0; t < n_threads && e == cudaSuccess; t++) {
        e = cudaStreamCreateWithFlags(&st[t], cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaMalloc(&work[t], std::max<size_t>(wb, 256));
    }
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    const int width = 2 * body;
    const size_t isz = (flags & MFDN_REQ_U16) ? 2 : 4;
    const auto t0 = std::chrono::steady_clock::now();
    if (e == cudaSuccess) {
        std::vector<std::thread> th;
        for (int t = 0; t < n_threads; t++)
            th.emplace_back([&, t]() {
                cudaSetDevice(c->device);
                for (int64_t lo = (int64_t)t * chunk; lo < n; lo += (int64_t)n_threads * chunk) {
                    const int64_t m = std::min<int64_t>(chunk, n - lo);
                    size_t w = wb;
                    const int32_t* rq = (const int32_t*)((const char*)d_req + (size_t)lo * width * isz);
                    const int r = body == 3 ? run<3>(c, m, rq, d_out + lo, d_mask ? d_mask + lo : nullptr, work[t], &w, flags, st[t])
                                            : run<2>(c, m, rq, d_out + lo, d_mask ? d_mask + lo : nullptr, work[t], &w, flags, st[t]);
                    if (r) { status[t] = r; break; }
                }
                if (cudaStreamSynchronize(st[t]) != cudaSuccess && status[t] == MFDN_OK) status[t] = MFDN_ERR_CUDA;
            });
        for (auto& x : th) x.join();
    }
    *seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    for (int t = 0; t < n_threads; t++) {
        if (work[t]) cudaFree(work[t]);
        if (st[t]) cudaStreamDestroy(st[t]);
    }
    if (e != cudaSuccess) return cuda_fail(c, e, "mfdn_multi_client setup");
    for (int t = 0; t < n_threads; t++)
        if (status[t]) return status[t] == MFDN_ERR_CUDA ? fail(c, MFDN_ERR_CUDA, "mfdn_multi_client: stream failed") : status[t];
    return MFDN_OK;
}

// The paper's wrapper over a ring of HOST_STREAMS buffers: chunk k uses stream k % HOST_STREAMS.  A stream runs its
// H2D copy, kernels and D2H copies in order, so with two streams the link idles while a stream computes (measured 21.1 ms
// for 2^26 compact requests); four keep both directions of the link busy.
extern "C" int mfdn_mscheme_host(mfdn_ctx* c, int body, int64_t n, const int32_t* h_req, double* h_out, uint8_t* h_mask,
                                 void* d_work, size_t* work_bytes, uint32_t flags, int64_t chunk)
{
    if (!c || !work_bytes || (body != 2 && body != 3) || n < 0 || chunk < 0) return c ? fail(c, MFDN_ERR_ARG, "bad argument") : MFDN_ERR_ARG;
    if (chunk == 0) chunk = 1 << 22;
    if (chunk > n && n > 0) chunk = n;
    const int width = 2 * body;
    const size_t isz = (flags & MFDN_REQ_U16) ? 2 : 4;   // bytes per SPS index of a request
    size_t inner = 0;
    int rc = body == 3 ? run<3>(c, chunk, nullptr, nullptr, nullptr, nullptr, &inner, flags, nullptr)
                       : run<2>(c, chunk, nullptr, nullptr, nullptr, nullptr, &inner, flags, nullptr);
    if (rc) return rc;
    const size_t b_req = align256((size_t)chunk * width * isz), b_out = align256((size_t)chunk * 8), b_mask = align256((size_t)chunk);
    const size_t per = b_req + b_out + b_mask + align256(inner);
    if (!d_work) { *work_bytes = HOST_STREAMS * per; return MFDN_OK; }
    if (*work_bytes < HOST_STREAMS * per) return fail(c, MFDN_ERR_OOM, "scratch too small");
    if (n == 0) return MFDN_OK;
    if (!h_req || !h_out) return fail(c, MFDN_ERR_ARG, "null host pointer");
    MFDN_CUDA(c, cudaSetDevice(c->device));
    for (int k = 0; k < HOST_STREAMS; k++)
        if (!c->hs[k]) MFDN_CUDA(c, cudaStreamCreateWithFlags(&c->hs[k], cudaStreamNonBlocking));
    auto drain = [&]() {
        cudaError_t first = cudaSuccess;
        for (int k = 0; k < HOST_STREAMS; k++) {
            const cudaError_t e = cudaStreamSynchronize(c->hs[k]);
            if (first == cudaSuccess) first = e;
        }
        return first;
    };
    int64_t k = 0;
    for (int64_t lo = 0; lo < n; lo += chunk, k++) {
        int64_t m = std::min<int64_t>(chunk, n - lo);
        cudaStream_t st = c->hs[k % HOST_STREAMS];
        char* base = (char*)d_work + (k % HOST_STREAMS) * per;
        int32_t* dreq = (int32_t*)base;
        double* dout = (double*)(base + b_req);
        uint8_t* dmask = (uint8_t*)(base + b_req + b_out);
        void* dw = base + b_req + b_out + b_mask;
        size_t wb = align256(inner);
        // on any failure: no copy may still be in flight on the caller's buffers when the call returns
        cudaError_t e = cudaMemcpyAsync(dreq, (const char*)h_req + (size_t)lo * width * isz, (size_t)m * width * isz, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) {
            rc = body == 3 ? run<3>(c, m, dreq, dout, dmask, dw, &wb, flags, st) : run<2>(c, m, dreq, dout, dmask, dw, &wb, flags, st);
            if (rc) { drain(); return rc; }
            e = cudaMemcpyAsync(h_out + lo, dout, (size_t)m * 8, cudaMemcpyDeviceToHost, st);
        }
        if (e == cudaSuccess && h_mask) e = cudaMemcpyAsync(h_mask + lo, dmask, (size_t)m, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) { drain(); return cuda_fail(c, e, "mfdn_mscheme_host copy"); }
    }
    const cudaError_t e0 = drain();
    if (e0 != cudaSuccess) return cuda_fail(c, e0, "cudaStreamSynchronize");
    return MFDN_OK;
}
