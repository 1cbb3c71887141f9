// NEXT-3 (SURVEY 8(e) / 8(f); PAPER.md:206 "overlap communication with computation", :291-295 strong scaling):
// the per-rank task and message schedule of the tile Cholesky over R GPUs of one NVSwitch domain.  HOST LOGIC ONLY --
// this file builds the lists; the single-GPU launch sequence of api.cu is what runs today.
//
// Distribution: tile ROW i belongs to rank i mod R (1D block-cyclic).  Column k, on every rank, over the rows it owns:
//     N(k)   newest term on the rows below the diagonal tile          needs L(k, k-1)            (message B, below)
//     O(k+1) older terms of column k+1                                needs row k+1 of L, columns < k   (message C of columns < k)
//     T(k)   X = S M_k^T and the quantising store                     needs M_k = inv(L_kk)      (message A)
// and on the owner of row k only: the diagonal chain of tile (k, k) and the inverse M_k.
// Messages (all in STORAGE precision, "conversion at the sender"; images are rebuilt by the receiver):
//     A(k)  M_k (FP16 hi / lo images, 4 nb^2 bytes)        owner(k)   -> all      on the critical path of T(k)
//     B(k)  tile (k+1, k)                                  owner(k+1) -> all      on the critical path of N(k+1) and of chain(k+1)
//     C(k)  the other tiles (i, k), i > k+1, of column k   all-gather             needed by O(i) / N(i) when row i becomes the
//                                                                                 B operand: at least one column of slack
#pragma once
#include <stdint.h>

#include <vector>

namespace krr {

enum DistOp : int32_t {
    DIST_CHAIN = 1,     // diagonal-tile chain + inverse of column k           (rank = owner(k))
    DIST_NEWEST = 2,    // N(k) on the rows [row list] of this rank
    DIST_OLDER = 3,     // O(k+1): arg = k + 1
    DIST_TRSM = 4,      // T(k)
    DIST_BCAST_M = 5,   // message A(k): root = owner(k)
    DIST_BCAST_NEXT = 6,// message B(k): root = owner(k + 1)
    DIST_ALLGATHER = 7  // message C(k): every rank contributes its tiles (i, k), i > k + 1
};

struct DistTask {
    int32_t op, k, root, nrows;     // nrows: tile rows of this rank the task covers (compute) / tiles this rank sends (C)
    int64_t bytes;                  // message size received by a rank (A, B, C), 0 for compute
};

inline int dist_owner(int i, int R) { return i % R; }

// rows i in (lo, NT) owned by `rank`
inline int dist_rows_owned(int lo_exclusive, int NT, int R, int rank) {
    int c = 0;
    for (int i = lo_exclusive + 1; i < NT; ++i) c += (dist_owner(i, R) == rank);
    return c;
}

// The schedule of one rank, in issue order.  tile_bytes(i, j): storage bytes of tile (i, j) from the precision map.
template <typename TileBytes>
inline void dist_build_schedule(int NT, int nb, int R, int rank, TileBytes tile_bytes, std::vector<DistTask>* out) {
    out->clear();
    const int64_t m_bytes = 4ll * nb * nb;                                  // hi + lo FP16 images of M_k
    for (int k = 0; k < NT; ++k) {
        const int below = dist_rows_owned(k, NT, R, rank);                  // own rows i > k
        // newest term (column k-1) on the own rows below the diagonal tile; the diagonal tile's share is part of the chain
        if (k >= 1 && below > 0) out->push_back({DIST_NEWEST, k, -1, below, 0});
        // older terms of column k+1, beside the chain of column k (lookahead)
        if (k >= 1 && k + 1 < NT) {
            const int rows = dist_rows_owned(k, NT, R, rank);               // own rows i >= k+1
            if (rows > 0) out->push_back({DIST_OLDER, k + 1, -1, rows, 0});
        }
        if (dist_owner(k, R) == rank) out->push_back({DIST_CHAIN, k, rank, 1, 0});
        if (k + 1 == NT) break;
        out->push_back({DIST_BCAST_M, k, dist_owner(k, R), 0, m_bytes});
        if (below > 0) out->push_back({DIST_TRSM, k, -1, below, 0});
        out->push_back({DIST_BCAST_NEXT, k, dist_owner(k + 1, R), 0, static_cast<int64_t>(tile_bytes(k + 1, k))});
        if (k + 2 < NT) {
            int64_t total = 0;
            int mine = 0;
            for (int i = k + 2; i < NT; ++i) {
                total += static_cast<int64_t>(tile_bytes(i, k));
                mine += (dist_owner(i, R) == rank);
            }
            out->push_back({DIST_ALLGATHER, k, -1, mine, total});
        }
    }
}

}  // namespace krr
