"""Pins for the oracle's basis / index maps (O1): counting identities, brute force,
rank(unrank(k)) = k for every state up to N = 20, the paper's CLT worked example (L175) and
table sizes (L185, Table 4).  CPU only."""
import math

import numpy as np
import pytest

from oracle import ftlm_oracle as fo
from oracle import c_oracle as co


def test_sector_dimensions_sum_to_full_space():
    for N in (1, 2, 5, 12, 16):
        dims = [fo.sector_basis(N, k).shape[0] for k in range(N + 1)]
        assert dims == [math.comb(N, k) for k in range(N + 1)]
        assert sum(dims) == 2 ** N


def test_basis_is_ascending_and_has_right_popcount():
    b = fo.sector_basis(14, 6)
    assert (np.diff(b.astype(np.int64)) > 0).all()
    assert (fo.popcount(b) == 6).all()


def test_rank_is_number_of_smaller_labels_bruteforce():
    # the definition itself, by brute force over the whole label space, N <= 12
    for N, N_up in ((6, 3), (9, 2), (12, 6), (12, 11), (7, 0), (7, 7)):
        labels = [n for n in range(2 ** N) if bin(n).count("1") == N_up]
        for n in range(2 ** N):
            expect = sum(1 for m in labels if m < n) if bin(n).count("1") == N_up else -1
            assert fo.rank_by_counting(n, N, N_up) == expect


def test_rank_unrank_roundtrip_every_state_up_to_N20():
    # rank(unrank(k)) = k over every state (all sectors) for N <= 20, Algorithm 1 + inverse
    for N in (1, 2, 3, 8, 13, 20):
        _, Dc = fo.cr_tables(N)
        for N_up in range(N + 1):
            D = math.comb(N, N_up)
            k = np.arange(D, dtype=np.int64)
            x = fo.alg1_unrank_vec(k, N, N_up, Dc)
            assert (fo.popcount(x) == N_up).all()
            assert (fo.alg1_rank_vec(x, N, N_up, Dc) == k).all()
            if D > 1:
                assert (np.diff(x.astype(np.int64)) > 0).all()   # ascending-label order (L125)


def test_three_index_maps_agree():
    # sorted search == counting definition == Algorithm 1 == CLT (Algorithm 2), in-sector and out
    N, N_up = 14, 5
    basis = fo.sector_basis(N, N_up)
    _, Dc = fo.cr_tables(N)
    M, Cb = fo.clt_build(basis, N)
    all_labels = np.arange(2 ** N, dtype=np.uint64)
    srt = fo.index_of_sorted(basis, all_labels)
    clt = fo.clt_lookup_vec(all_labels, M, Cb)
    assert (srt == clt).all()
    assert (srt[basis.astype(np.int64)] == np.arange(basis.shape[0])).all()
    assert (srt[fo.popcount(all_labels) != N_up] == -1).all()
    a1 = fo.alg1_rank_vec(basis, N, N_up, Dc)
    assert (a1 == np.arange(basis.shape[0])).all()
    rng = np.random.default_rng(0)
    for n in rng.integers(0, 2 ** N, size=300):
        n = int(n)
        assert fo.rank_by_counting(n, N, N_up) == srt[n] == fo.clt_lookup(n, M, Cb)
        if srt[n] >= 0:
            assert fo.alg1_rank(n, N, N_up, Dc) == srt[n]
            assert fo.unrank_by_counting(int(srt[n]), N, N_up) == n


def test_cr_tables_are_binomials_at_spin_half():
    # Eq. 15 with d = 2 is Pascal's rule; reading 25: D_c(p,A,0) = 0, D_c(p,A,1) = C(p,A)
    D, Dc = fo.cr_tables(18)
    for m in range(19):
        for A in range(19):
            assert D[m][A] == (math.comb(m, A) if A <= m else 0)
            assert Dc[m][A][0] == 0 and Dc[m][A][1] == D[m][A]


def test_cr_tables_general_spin_dimension():
    # Eq. 15 for s = 1 (d = 3): D(12, 12) is the M=0 dimension of the s=1 icosahedron, Table 1
    D, _ = fo.cr_tables(12, two_s=2)
    assert D[12][12] == 73789          # PAPER.md Table 1, row s = 1 (L89)


def test_clt_worked_example_L175(golden_paper):
    g = golden_paper
    members = [int(s) for s in g["clt_example_members"].split(",")]
    N, blk = 7, 2                       # any block; labels 32*blk + j
    basis = np.array(sorted(32 * blk + j for j in members), dtype=np.uint64)
    M, C = fo.clt_build(np.concatenate([np.array([3, 40], dtype=np.uint64), basis]), N)
    assert int(M[blk]) == int(g["clt_example_mask"], 2)
    j = int(g["clt_example_query_j"])
    assert (int(M[blk]) & ((1 << j) - 1)) == int(g["clt_example_masked"], 2)
    assert fo.clt_lookup(32 * blk + j, M, C) == int(C[blk]) + int(g["clt_example_local_rank"])
    assert int(C[blk]) == 2             # two in-sector labels (3, 40) in preceding blocks: Eq. 18
    assert fo.clt_lookup(32 * blk + 1, M, C) == -1      # Alg. 2 step 2
    assert fo.clt_lookup(32 * blk + 0, M, C) == int(C[blk])   # j = 0: (2^0 - 1) = 0 (reading 21)


def test_clt_and_memory_sizes_from_paper(golden_paper):
    g = golden_paper
    assert fo.clt_bytes(30) == int(g["clt_bytes_N30"])
    assert 4 * 2 ** 30 == int(g["full_table_bytes_N30"])
    assert int(g["full_table_bytes_N30"]) // fo.clt_bytes(30) == int(g["clt_reduction"])
    D0 = math.comb(30, 15)
    assert D0 == int(g["table4_D0"])
    assert round(4 * D0 / 1e6) == int(g["table4_basis_MB"])
    assert abs(3 * 4 * 4 * D0 / 1e6 - int(g["table4_vectors_MB_B4"])) < 10   # paper rounds to 10 MB


def test_nnz_formula_table1(golden_paper):
    assert math.comb(12, 6) == int(golden_paper["table1_D0"])
    assert fo.nnz_formula(12, 6, 30) == int(golden_paper["table1_Nnz"])


def test_c_oracle_basis_and_search_match_numpy():
    for N, N_up in ((10, 5), (17, 8), (20, 3)):
        b_np = fo.sector_basis(N, N_up)
        b_c = co.enumerate_basis(N, N_up)
        assert (b_np == b_c).all()
        rng = np.random.default_rng(N)
        lab = rng.integers(0, 2 ** N, size=5000).astype(np.uint64)
        assert (co.index_many(b_c, lab) == fo.index_of_sorted(b_np, lab)).all()


def test_counting_rank_matches_enumeration_at_N30_samples():
    # the counting definition (used for sampled checks at N = 34) against the explicitly
    # enumerated + sorted basis at N = 26 (66 MB), on random and edge rows
    N, N_up = 26, 13
    basis = co.enumerate_basis(N, N_up)
    D = basis.shape[0]
    rng = np.random.default_rng(5)
    rows = np.concatenate([[0, 1, D - 2, D - 1], rng.integers(0, D, size=400)])
    for t in rows:
        n = int(basis[int(t)])
        assert fo.rank_by_counting(n, N, N_up) == int(t)
        assert fo.unrank_by_counting(int(t), N, N_up) == n


def test_lin_two_table_map_equals_sorted_search_on_every_label():
    """SURVEY 8(f)-3 / PAPER.md L119: Lin's two half-system tables (built by counting over the explicit basis) give the
    ascending-order index of every in-sector label and -1 outside, for every sector of N = 9 (odd: halves 4 + 5), 12
    and 13; table sizes are 2^(N - N//2) and 2^(N//2)."""
    for N in (9, 12, 13):
        all_labels = np.arange(1 << N, dtype=np.uint64)
        for n_up in range(N + 1):
            basis = fo.sector_basis(N, n_up)
            h, Ja, Jb = fo.lin_tables(basis, N)
            assert (h, Ja.shape[0], Jb.shape[0]) == (N // 2, 1 << (N - N // 2), 1 << (N // 2))
            got = fo.lin_lookup_vec(all_labels, N, n_up, h, Ja, Jb)
            assert (got == fo.index_of_sorted(basis, all_labels)).all()
    # brute force on one sector: the index is the number of smaller sector labels
    basis = fo.sector_basis(10, 4)
    h, Ja, Jb = fo.lin_tables(basis, 10)
    for n in basis[::7]:
        assert fo.lin_lookup_vec([n], 10, 4, h, Ja, Jb)[0] == fo.rank_by_counting(int(n), 10, 4)


def test_c_oracle_under_ubsan(tmp_path):
    """SURVEY section 5 ("ASan/UBSan on oracle"): the C oracle compiled with -fsanitize=undefined,bounds (trap on error)
    must run its whole interface - enumeration, search, H.v, neighbour lists, Lanczos - on small sectors (incl. the
    one-state sectors and N = 34 labels) without tripping, and agree with the numpy oracle."""
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    so = str(tmp_path / "liborc_ubsan.so")
    subprocess.check_call(["gcc", "-O1", "-g", "-fopenmp", "-shared", "-fPIC", "-fsanitize=undefined,bounds",
                           "-fsanitize-undefined-trap-on-error", os.path.join(root, "oracle", "ftlm_oracle_c.c"), "-o", so, "-lm"])
    code = ("import sys; sys.path.insert(0, %r)\n"
            "import numpy as np\n"
            "from oracle import c_oracle as co, ftlm_oracle as fo\n"
            "from paper_2605_26261_b200 import workloads as W\n"
            "for w, n_up in ((W.ring(12, 1.0, 0.5), 6), (W.ring(9), 0), (W.ring(9), 9), (W.icosahedron(), 7)):\n"
            "    basis = co.enumerate_basis(w.N, n_up)\n"
            "    assert (basis == fo.sector_basis(w.N, n_up)).all()\n"
            "    v = np.random.default_rng(1).standard_normal(basis.shape[0])\n"
            "    y = co.apply_rows(w.N, w.bond_i, w.bond_j, w.J, 0.2, n_up, basis, v)\n"
            "    assert np.abs(y - fo.apply_H(basis, w.N, w.bond_i, w.bond_j, w.J, 0.2, n_up, v)).max() < 1e-12\n"
            "    nb = co.neighbors_rows(w.N, w.bond_i, w.bond_j, basis, np.arange(basis.shape[0], dtype=np.int64))\n"
            "    assert (nb == fo.neighbor_indices(basis, w.bond_i, w.bond_j, np.arange(basis.shape[0]))).all()\n"
            "    a, b = co.lanczos(w.N, w.bond_i, w.bond_j, w.J, 0.0, n_up, basis, fo.start_vector(3, n_up, 0, basis.shape[0]), 10)[:2]\n"
            "    assert np.isfinite(a).all() and np.isfinite(b).all()\n"
            "lab = np.array([(1 << 34) - 1 - (1 << 20), (1 << 17) - 1, 5], dtype=np.uint64)\n"
            "assert (co.index_many(co.enumerate_basis(20, 3), np.array([7, 11, 1 << 19], dtype=np.uint64)) == [0, 1, -1]).all()\n"
            "print('ok')\n" % root)
    p = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600, env=dict(os.environ, FTLM_ORACLE_LIB=so))
    assert p.returncode == 0 and p.stdout.strip().endswith("ok"), (p.returncode, p.stderr[-1500:])
