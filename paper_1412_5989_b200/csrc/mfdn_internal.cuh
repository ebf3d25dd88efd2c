// Internal layout of the device tables (N0) shared by the host API and the kernels.
// Not part of the ABI.  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <atomic>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/mfdn_b200.h"

namespace mfdn {

// ---- SPS record (A0): one 32-bit word per single-particle state -------------------------------
//  [0,10) orbital   [10,17) im = (2m+2j)/2   [17,24) 2j   [24,26) tz bit (1 <=> 2tz = +1)   [26,28) l & 1
// The fields above bit 10 are two bits wider than their values: (r0 >> 10) + (r1 >> 10) + (r2 >> 10) is the packed
// sum of every field over up to three particles (M, Tz and parity conservation from one addition).  e = 2n+l is
// not kept: S5 (sum of e <= E3max) is implied by S6 (the tuple is listed), because the upload rejects listed
// states above E3max.
__host__ __device__ inline uint32_t sps_pack(int orb, int im, int tzbit, int twoj, int lpar)
{
    return (uint32_t)orb | ((uint32_t)im << 10) | ((uint32_t)twoj << 17) | ((uint32_t)tzbit << 24) | ((uint32_t)lpar << 26);
}
__host__ __device__ inline int rec_orb(uint32_t r) { return r & 1023; }
__host__ __device__ inline int rec_im(uint32_t r) { return (r >> 10) & 31; }
__host__ __device__ inline int rec_twoj(uint32_t r) { return (r >> 17) & 31; }
__host__ __device__ inline int rec_tz(uint32_t r) { return (r >> 24) & 1; }
__host__ __device__ inline int rec_lpar(uint32_t r) { return (r >> 26) & 1; }
// fields of a packed sum (r0 >> 10) + (r1 >> 10) [+ (r2 >> 10)]
__host__ __device__ inline int sum_im(uint32_t s) { return s & 127; }
__host__ __device__ inline int sum_twoj(uint32_t s) { return (s >> 7) & 127; }
__host__ __device__ inline int sum_tz(uint32_t s) { return (s >> 14) & 3; }
__host__ __device__ inline int sum_lpar(uint32_t s) { return (s >> 16) & 3; }

constexpr int MAX_TWOJ = 21;       // 3*MAX_TWOJ <= 63 so that (2J,2T) fits a 64-bit channel mask
constexpr int NISO3 = 5;           // isospin slots per 3-body cell: (T12,T12',T) = (0,0,1/2) (0,1,1/2) (1,0,1/2) (1,1,1/2) (1,1,3/2)
constexpr int NBIN3 = 20;          // isospin bins: (bra tz pattern, ket tz pattern) pairs with equal MT
constexpr int CELL2 = 2;           // doubles per 2-body slab cell: T = 0, 1 (16 B)
constexpr uint32_t NO_SLAB = 0xFFFFFFFFu;
constexpr int CG_GUARD = 8192;     // zero doubles before and after the stage-2 table (see Tables::cg2g)

// 3-body slab of a (bra tuple, ket tuple) group = NISO3 isospin planes of `gsize` doubles each; inside a plane the
// cells are in the order the kernel's loops read them:
//   for J (common range, ascending) / for bra J12 in range(J) / for ket J12' in range(J)
// one "row" = the nk(J) cells of a fixed (J, J12), padded to an even count (16-byte units), zero where a state is
// not listed.  The isospin-combined copy Vw = sum_s w[s] * plane[s] that the transform stages in shared memory has
// the same indexing.
__host__ __device__ inline int row_pitch3(int nk) { return (nk + 1) & ~1; }
constexpr int HOST_STREAMS = 4;    // internal streams / chunk buffers of mfdn_mscheme_host
constexpr int ITEM3 = 512;         // max records per work item of the 3-body transform (one group per item)
// Isospin-combined slabs (A2): for every group and every isospin bin the weighted plane sum Vw[cell] =
// sum_s w[bin][s] * plane_s[cell], precomputed at upload so that staging it is a pure bulk copy.  The two 32-bit
// halves of a value live in separate word planes: bin b occupies vw_stride(gsize) 32-bit words, low words at
// [0, gsize), high words at [gsize, 2*gsize), one pad word.  The stride is ODD, so the 20 bins of one cell fall
// into 20 different shared-memory banks: a warp whose lanes sit in any mixture of bins reads a cell with two
// conflict-free 32-bit loads (measured: 2.0 cycles per cell against 3.7 for 64-bit loads over 20 random bins).
// With MFDN_OPT_SLAB_FP32 a value is ONE fp32 word (footprint variant, NEXT-4): bin b occupies gsize | 1 words (odd again).
__host__ __device__ inline uint32_t vw_stride(uint32_t gsize, int f32 = 0) { return f32 ? (gsize | 1u) : 2u * gsize + 1u; }
constexpr int DENSE_CAP = 1024;    // doubles of one (group, M, bin) block of the dense path, both dimensions padded to 8 (one warp's tile buffer)
constexpr int DENSE_RMAX = 64;     // flattened ket rows (J, J12') of a group on the dense path
constexpr int VW_WORDS = 5120;     // 32-bit words of one staged slab (20 KB): all 20 bins of a group with gsize <= 127
constexpr uint32_t ZERO_ITEM = 0xFFFFFFFFu;   // work item whose records all have value 0 (no slab / failed S1-S6)
constexpr uint32_t STOP_ITEM = 0xFFFFFFFEu;   // posted by the producer warp of k_transform3 after its last item

// ---- packed canonical request record (H1 output), 64 bit --------------------------------------------
// 2-body: [0,30) im of the canonical particles (5 bits each: bra at 0,5; ket at 15,20)   [30,36) tz bits (bra then ket)
//         [36] 1 = odd permutation (sign -1)                     [37,64) group key, REC_INVALID if S1-S6 fail
// 3-body: [0,12) sigma_b  [12,24) sigma_k : index of the bra / ket m-state in its tuple's coefficient table (M-major)
//         [24,29) isospin bin   [29] 1 = odd permutation   [30,36) iM = ima+imb+imc of the bra (M = iM - (ja+jb+jc)/2)
//         [37,64) sort key: 2-body bra_tuple*n_tup+ket_tuple; 3-body the (group, M) bucket gbase3[group] + iM - iMmin
constexpr unsigned REC_KEY_SHIFT = 37;
constexpr uint32_t REC_INVALID = 0x7FFFFFFu;
constexpr int MAX_STATES3 = 4096;   // (ja+1)(jb+1)(jc+1) of a tuple must fit the 12-bit sigma fields

// ---- per-tuple descriptor (A2), 16 bytes ---------------------------------------------------------
// 3-body: x = ja | jb<<8 | jc<<16 | (a==b)<<24 | par<<25      (ja.. are 2j)
//         y = J12min | J12max<<8 | twoJmin<<16 | twoJmax<<24
//         z = offset of the tuple's state masks in stmask3 (entries: [J12-J12min][T12], suffix-ORed over J12)
//         w = start of the tuple's sigma table in sig3 (during the upload: offset of the tuple's row map)
// tk3 (what the transform kernel needs of a tuple): x = offset of the tuple's coefficient table in dtab3 (doubles),
//         y = its m-state count S = (ja+1)(jb+1)(jc+1), z = first entry of the tuple in jinfo3,
//         w = (ja+jb+jc) | twoJmin<<16 | twoJmax<<24
// 2-body: x = ja | jb<<8 | (a==b)<<24 | par<<25,  y = Jmin | Jmax<<8,  z = state mask (low), w = (high)
struct Tables {
    // A0
    const uint32_t* sps_rec;
    int n_sps, n_orb;
    // A1: CG tables.  nj = number of half-integer j values (2j = 1,3,..,2*nj-1)
    int nj;
    const double* cg1;       // stage 1 blocks [(2j1-1)/2 * nj + (2j2-1)/2]
    const int32_t* cg1_off;
    const double* cg2;       // stage 2 blocks [J12 * nj + (2j-1)/2],  J12 = 0..2*nj-1
    const int32_t* cg2_off;
    const double* cg2g;      // = cg2 - CG_GUARD: row-table offsets are relative to this, so that a lane whose
                             // |M12| > J12 (stage-1 factor = 0) still reads valid, finite memory
    const double* wtab3;     // [64][6] isospin weights w[5] (+pad) indexed by the 6 tz bits of a record
    const double* wtab2;     // [16][2]
    const double* wbin3;     // [NBIN3][NISO3] the same weights indexed by isospin bin
    const uint8_t* tz2bin3;  // [64] tz bits of a record -> isospin bin
    double iso3[8][3];       // [ta<<2|tb<<1|tc][(T12,T) = (0,1/2),(1,1/2),(1,3/2)]
    double iso2[4][2];       // [ta<<1|tb][T]
    // A2, 3-body
    int n_tup3, e3max;
    const int32_t* tuple_id3;      // [n_orb^3] -> tuple or -1
    const int2* ab3;               // [n_orb^2] {first tuple of (a,b,*), cmin | count<<16} if every (a,b) has a dense c range, else NULL
    const int4* tdesc3;
    const uint4* sgrp3;            // [n_tup3^2] {start of the group's slab in 16-byte units or NO_SLAB, doubles per plane,
                                   //              start of its isospin-combined slabs in vw20 in 16-byte units,
                                   //              dense-block path feasible << 31 | (bra, ket) m-state pairs with equal M}
    const uint32_t* gbase3;        // [n_tup3^2 + 1] first (group, M) bucket of a group; same-parity groups own
                                   //              min(ja+jb+jc, jd+je+jf) + 1 buckets (one per common M), the others none
    const uint32_t* rowbase3;      // [n_tup3] and
    const uint16_t* colcum3;       // [ncls3][n_tup3]: gbase3[b][k] = rowbase3[b] + colcum3[class(b)][k], class(b) = bits 26..30 of
    int ncls3;                     //              tdesc3[b].x (distinct (ja+jb+jc, parity) of the tuples); ncls3 = 0: not available
    int sig_len3, stmask_len3;     // entries of sig3 and of stmask3
    uint32_t n_buckets3;           // = gbase3[n_tup3^2]; bucket n_buckets3 collects the requests failing S1-S6
    const double* slab3;
    const uint32_t* vw20;          // isospin-combined slabs, split word planes (see vw_stride)
    int vw_f32;                    // 1: the slabs hold fp32 values, one word each (MFDN_OPT_SLAB_FP32)
    const unsigned long long* stmask3;
    const unsigned long long* stm12_3;   // S7 by direct look-up: [stm12_off3[tuple] + (ima + imb) * 2 + (MT12 == 0)] = channels (J, T) in which the
    const int32_t* stm12_off3;           // tuple has a listed state with J12 >= |M12| and a T12 admissible for MT12 (built from stmask3 at upload)
    int stm12_len3;
    const int4* tk3;               // [n_tup3] see above
    const int2* jinfo3;            // per (tuple, J): {offset of the J block in the tuple's coefficient table (doubles, even), rows nb(J)}
    const double* dtab3;           // per tuple and J block [sigma][row] = <ja ma jb mb|J12 M12> <J12 M12 jc mc|J M>, rows = J12 ascending
    const uint16_t* mstart3;       // per tuple (at mstoff3[tuple]): first sigma of every iM, sumj + 2 entries (M-major order of the m-states)
    const int32_t* mstoff3;
    const uint16_t* sig3;          // per tuple [(ima*(jb+1)+imb)*(jc+1)+imc] -> sigma: m-states ordered by (M, ima, imb), so that
                                   // requests with equal M (bra and ket always have equal M) read neighbouring entries
    const uint16_t* isig3;         // inverse of sig3 (same offsets): sigma -> (ima*(jb+1)+imb)*(jc+1)+imc
    const int4* torb3;             // [n_tup3] orbitals {a, b, c, -} of a tuple
    const int32_t* spsidx3;        // [(orbital*2 + tz bit)*32 + m index] -> SPS index or -1
    // A2, 2-body
    int n_tup2;
    const int32_t* tuple_id2;      // [n_orb^2]
    const int4* tdesc2;
    const uint32_t* slab_off2;
    const double* slab2;
    unsigned long long* bad_count;
};

}  // namespace mfdn

struct mfdn_ctx {
    int device = 0;
    int stage = 0;  // 1 orbitals, 2 cg built
    bool has2 = false, has3 = false;
    bool opt_slab_fp32 = false;   // mfdn_option(MFDN_OPT_SLAB_FP32), read by mfdn_coupled_upload_3b
    std::string err;            // last error message; guarded by `mu` (mfdn_last_error hands out a per-thread copy)
    std::mutex mu;              // guards err, ev_pending, ev_pool: mscheme_* may be called from several host threads
    mfdn::Tables t{};
    int tjmax = 0;
    // host copies
    std::vector<int32_t> orb_n, orb_l, orb_twoj, h_cg2_off;
    std::vector<uint32_t> h_sps_rec;
    // host copies for sizing the blocks of mfdn_mscheme_blocks_3b
    std::vector<int32_t> h_tuple_id3, h_mstoff3;
    std::vector<int4> h_tdesc3;
    std::vector<uint16_t> h_mstart3;
    std::vector<uint4> h_sgrp3;
    std::vector<void*> owned;  // device allocations
    int64_t n_cg1 = 0, n_cg2 = 0;
    int64_t slab_bytes2 = 0, slab_bytes3 = 0, dtab_bytes3 = 0, vw_bytes3 = 0;
    std::atomic<int64_t> launches{0};
    int num_sms = 148;
    std::atomic<bool> keys_attr_set{false};  // same for k_keys3s
    std::atomic<bool> part_attr_set{false};  // dynamic shared-memory limit of the partition kernels raised (first sort-path call)
    std::atomic<int> tr_blocks_per_sm{0};   // resident k_transform3 blocks per SM (occupancy query at the first call)
    // measurement hooks
    bool profile = false;
    struct EvTriple { cudaEvent_t a, b, d, c; bool has_sort; };   // start | transform kernel start | its end | end of call
    std::vector<EvTriple> ev_pending;
    std::vector<cudaEvent_t> ev_pool;
    // host-buffer wrapper
    cudaStream_t hs[4] = {nullptr, nullptr, nullptr, nullptr};
};

namespace mfdn {
int fail(mfdn_ctx* c, int code, const std::string& msg);
int cuda_fail(mfdn_ctx* c, cudaError_t e, const char* what);
}  // namespace mfdn

#define MFDN_CUDA(ctx, call)                                                  \
    do {                                                                      \
        cudaError_t e__ = (call);                                             \
        if (e__ != cudaSuccess) return mfdn::cuda_fail((ctx), e__, #call);    \
    } while (0)
