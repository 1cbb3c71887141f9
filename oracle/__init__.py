"""CPU oracle for the mixed-precision tile Cholesky of K + lambda*I (paper's Associate phase).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only `tests/`, `__graft_entry__.smoke()` and the
`cpu_baseline` / `--impl reference` legs of `bench.py` may import this package.  It shares no
code with `paper_2409_01712_b200/` (the CUDA path) and never imports it; the only module both
sides use is `krr_inputs` (seeded synthetic inputs, none of the method's arithmetic).

What it computes, and where the paper defines it (citations are PAPER.md lines):

* `oracle.cholesky.tile_cholesky_fp64`   -- FACTORIZE(K + alpha*Id), Alg. 3 l.3, the
  textbook tile POTRF/TRSM/SYRK/GEMM algorithm the paper names, in FP64.
* `oracle.cholesky.tile_cholesky_emulated` -- the "tiled mosaic of precisions embedded in a single
  stored copy of the matrix" with FP32/FP16/FP8-E4M3 tiles,
  software rounding, FP64 arithmetic between the rounding points fixed in DESIGN.md (readings
  R3-R7).
* `oracle.precision_map.precision_map`   -- tile-centric adaptive precision applied to the
  off-diagonal tiles at the start of Associate; the rule text is
  BASELINE.json's (the paper prints no formula; reading R1).
* `oracle.solve.potrs_fp64`              -- Solve(K~, P_h), Alg. 3 l.5, forward and
  backward substitution.

* `oracle.build_phase`                    -- Build (Alg. 2 with the Gaussian kernel of Alg. 5, PAPER.md:92-106,
  :136-143) and Predict (Alg. 4, :116-122) by their definitions in exact integers / FP64, and the paper's MSPE
  (:243) and Pearson correlation (:262-266); pinned by the paper's three-patient example (:176-188), the
  D + D^T - 2 G G^T identity, scipy cdist, closed forms and numpy.corrcoef (tests/test_oracle_build.py).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): closed-form factors (diagonal, Lehmer, min(i,j),
equicorrelation, Kac-Murdock-Szego, hand 2x2/3x3), brute-force scalar Cholesky for n <= 64 and every
nb | n, LAPACK (numpy) Cholesky, invariants, exactly-representable constructions that every
precision map must reproduce bit for bit, numpy.float16 / torch.float8_e4m3fn casts and the full
E4M3 code table for the rounding emulators, threshold constructions for the map rule, and the
Sherman-Morrison closed form for the solve.  "Parity unpinned" items: none of the functions lacks a
pin; what nothing pins is any *number from the paper* -- PAPER.md prints no worked example, error
bound or rule formula for this path, so every pin is mathematical.
"""
