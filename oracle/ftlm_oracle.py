"""FP64 CPU oracle for the FTLM hot path of arxiv/paper_2605_26261.

TEST INFRASTRUCTURE ONLY.  This file is the plain, slow, obviously-correct statement of
what the CUDA path computes.  Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s
`cpu_baseline` / `--impl reference` legs may import it.  It shares no code, table or constant
generator with `paper_2605_26261_b200/` and imports nothing from it; every function cites the
passage of PAPER.md it restates.  Everything is float64 / Python int.

Conventions: spin-1/2 only (d = 2); bit k of a label = 1 <=> site k up
(Eq. 11); N_up = N/2 + M_z (Eq. 17); sector basis = ascending labels,
0-based index (L125, L154); index -1 = not in the sector (Alg. 2 step 2, L172).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): dimer and 4-ring closed-form spectra,
full-space Kronecker-product Hamiltonian for N <= 12, Table 1 N_nz = 16 044, sector-trace
closed form, [H, S^2] = 0, rank(unrank(k)) = k for every state up to N = 20, brute-force
"number of smaller labels", the L175 CLT worked example, Table 4 sizes, sum_k w_k = 1,
FTLM with R = D unit starts and N_L = D == exact Z, dimer C(T), chi(T) closed forms.
Parity unpinned: none of the functions below (see DESIGN.md section 5 for what pins what).
"""
from __future__ import annotations

import math

import numpy as np

# --------------------------------------------------------------------------------------
# O1  basis, index map
# --------------------------------------------------------------------------------------


def popcount(x):
    return np.bitwise_count(np.asarray(x, dtype=np.uint64)).astype(np.int64)


def sector_basis(N: int, N_up: int) -> np.ndarray:
    """All labels n in [0, 2^N) with popcount N_up, ascending (L103: "a basis array
    containing the integer labels of the sector basis states"; ordering L154).
    Explicit enumeration of the whole label space, in chunks."""
    out = []
    total = 1 << N
    step = 1 << min(N, 22)
    for lo in range(0, total, step):
        lab = np.arange(lo, lo + step, dtype=np.uint64)
        out.append(lab[np.bitwise_count(lab) == N_up])
    basis = np.concatenate(out)
    assert basis.shape[0] == math.comb(N, N_up)
    return basis  # already ascending


def index_of_sorted(basis: np.ndarray, labels) -> np.ndarray:
    """State-to-index map by binary search in the sorted basis (L119 lists search-based
    maps; this is the oracle's plain one).  -1 where the label is not in the sector."""
    labels = np.asarray(labels, dtype=np.uint64)
    pos = np.searchsorted(basis, labels)
    pos_c = np.minimum(pos, basis.shape[0] - 1)
    ok = basis[pos_c] == labels
    return np.where(ok, pos_c, -1).astype(np.int64)


def rank_by_counting(n: int, N: int, N_up: int) -> int:
    """Definition of the index: the number of sector labels strictly smaller than n
    (L154: basis ordered by increasing label).  Counted position by position: a label
    m < n first differs from n at some bit p where n has 1 and m has 0; the p lower
    bits of m are then free but must hold the ones still missing.  Returns -1 if n is not
    in the sector.  Python ints: exact at any N."""
    if n >> N or bin(n).count("1") != N_up:
        return -1
    cnt, ones_above = 0, 0
    for p in range(N - 1, -1, -1):
        if (n >> p) & 1:
            need = N_up - ones_above      # ones that the lower p bits of m must hold
            if 0 <= need <= p:
                cnt += math.comb(p, need)
            ones_above += 1
    return cnt


def unrank_by_counting(t: int, N: int, N_up: int) -> int:
    """Inverse of rank_by_counting: the t-th smallest label with popcount N_up.  At bit p
    with A ones still to place: the labels with bit p = 0 are the first C(p, A) ones
    (L136: "determines each digit by comparing the remaining rank with the cumulative
    counts"; tie rule = reading 26)."""
    assert 0 <= t < math.comb(N, N_up)
    n, A = 0, N_up
    for p in range(N - 1, -1, -1):
        c = math.comb(p, A) if 0 <= A <= p else 0
        if t >= c:
            n |= 1 << p
            t -= c
            A -= 1
    assert A == 0 and t == 0
    return n


# ---- Combinatorial ranking exactly as the paper writes it (Eqs. 15-17, Algorithm 1) -----


def cr_tables(N: int, two_s: int = 1):
    """D(m, A) by the recursion Eq. 15 (L121-L123) and the cumulative table
    D_c(m, A, a) = sum_{q<a} D(m, A-q) of Eq. 16 (L125-L128), for digits 0..2s."""
    Amax = N * two_s
    D = [[0] * (Amax + 1) for _ in range(N + 1)]
    D[0][0] = 1
    for m in range(1, N + 1):
        for A in range(Amax + 1):
            D[m][A] = sum(D[m - 1][A - q] for q in range(two_s + 1) if A - q >= 0)
    Dc = [[[sum(D[m][A - q] for q in range(a) if A - q >= 0) for a in range(two_s + 1)]
           for A in range(Amax + 1)] for m in range(N + 1)]
    return D, Dc


def alg1_rank(x: int, N: int, A_tot: int, Dc) -> int:
    """Algorithm 1 (L138-L144) with reading 23 (the lost minus signs restored):
    rank <- 0, A <- A_tot; for p = N-1..0: a_p = p-th digit; rank += D_c(p, A, a_p);
    A <- A - a_p."""
    rank, A = 0, A_tot
    for p in range(N - 1, -1, -1):
        a_p = (x >> p) & 1
        rank += Dc[p][A][a_p] if A >= 0 else 0
        A -= a_p
    return rank


def alg1_rank_vec(x, N: int, A_tot: int, Dc) -> np.ndarray:
    """Algorithm 1 on an array of labels (same steps, vectorised over labels only)."""
    x = np.asarray(x, dtype=np.uint64)
    tab = np.array([[Dc[p][A][1] for A in range(N + 1)] for p in range(N + 1)], dtype=np.uint64)
    rank = np.zeros(x.shape, dtype=np.uint64)
    A = np.full(x.shape, A_tot, dtype=np.int64)
    for p in range(N - 1, -1, -1):
        a_p = ((x >> np.uint64(p)) & np.uint64(1)).astype(np.int64)
        add = tab[p][np.clip(A, 0, N)]
        rank += np.where((a_p == 1) & (A >= 0), add, np.uint64(0))
        A -= a_p
    return rank.astype(np.int64)


def alg1_unrank_vec(t, N: int, A_tot: int, Dc) -> np.ndarray:
    """Inverse map with the same outer loop (L136), vectorised over indices."""
    t = np.asarray(t, dtype=np.uint64).copy()
    tab = np.array([[Dc[p][A][1] for A in range(N + 1)] for p in range(N + 1)], dtype=np.uint64)
    x = np.zeros(t.shape, dtype=np.uint64)
    A = np.full(t.shape, A_tot, dtype=np.int64)
    for p in range(N - 1, -1, -1):
        c = tab[p][np.clip(A, 0, N)]
        c = np.where(A >= 0, c, np.uint64(0))
        one = t >= c
        one &= A > 0
        x |= np.where(one, np.uint64(1) << np.uint64(p), np.uint64(0))
        t = np.where(one, t - c, t)
        A -= one.astype(np.int64)
    return x


# ---- Compressed lookup table exactly as the paper writes it (L148-L183) -----------------


def clt_build(basis: np.ndarray, N: int):
    """CLT construction, L183: one pass over the sorted basis sets bit (n mod 32) of
    M_{floor(n/32)}; prefix counts C_b = cumulative sum of block popcounts (Eq. 18).
    Last block zero-padded if 2^N is not a multiple of 32 (L181)."""
    nblk = max(1, ((1 << N) + 31) // 32)
    M = np.zeros(nblk, dtype=np.uint32)
    b = (basis >> np.uint64(5)).astype(np.int64)
    j = (basis & np.uint64(31)).astype(np.uint32)
    np.bitwise_or.at(M, b, (np.uint32(1) << j))
    pc = np.bitwise_count(M).astype(np.int64)
    C = np.concatenate([[0], np.cumsum(pc)[:-1]]).astype(np.int64)
    return M, C


def clt_lookup(n: int, M: np.ndarray, C: np.ndarray) -> int:
    """Algorithm 2 (L167-L173), reading 24: b = floor(n/32), j = n mod 32; -1 if bit j of
    M_b is zero; else C_b + popcount(M_b & (2^j - 1))  (Eqs. 19-20)."""
    b, j = n >> 5, n & 31
    Mb = int(M[b])
    if not (Mb >> j) & 1:
        return -1
    return int(C[b]) + bin(Mb & ((1 << j) - 1)).count("1")


def clt_lookup_vec(n, M: np.ndarray, C: np.ndarray) -> np.ndarray:
    n = np.asarray(n, dtype=np.uint64)
    b = (n >> np.uint64(5)).astype(np.int64)
    j = (n & np.uint64(31)).astype(np.uint32)
    Mb = M[b]
    inside = ((Mb >> j) & np.uint32(1)) == 1
    low = Mb & ((np.uint32(1) << j) - np.uint32(1))
    return np.where(inside, C[b] + np.bitwise_count(low).astype(np.int64), -1).astype(np.int64)


def lin_tables(basis: np.ndarray, N: int):
    """Lin's two-table index (L119: "partitioning the system into two halves, with rank tables of size approximately
    d^(N/2) for each half"), from the explicit basis in ascending order (L154): label n = (a << h) | b with
    h = N // 2 low positions; index(n) = Ja[a] + Jb[b].  Ja[a] = number of sector labels whose high half is smaller
    than a (labels with equal high half are contiguous); Jb[b] = position of b among the h-bit words of the same
    popcount in ascending order (the labels sharing a high half differ only in b and all have that popcount).
    Built by counting, not by a formula."""
    h = N // 2
    hi = (basis >> np.uint64(h)).astype(np.int64)
    Ja = np.concatenate(([0], np.cumsum(np.bincount(hi, minlength=1 << (N - h)))))[: 1 << (N - h)].astype(np.int64)
    words = np.arange(1 << h, dtype=np.uint64)
    pc = popcount(words)
    Jb = np.zeros(1 << h, dtype=np.int64)
    for k in range(h + 1):
        sel = np.flatnonzero(pc == k)                   # ascending
        Jb[sel] = np.arange(sel.shape[0])
    return h, Ja, Jb


def lin_lookup_vec(n, N: int, N_up: int, h: int, Ja: np.ndarray, Jb: np.ndarray) -> np.ndarray:
    """index = Ja[n >> h] + Jb[n & (2^h - 1)], -1 for labels outside the sector (two table reads and a popcount)."""
    n = np.asarray(n, dtype=np.uint64)
    ok = (popcount(n) == N_up) & ((n >> np.uint64(N)) == 0) if N < 64 else (popcount(n) == N_up)
    a = (n >> np.uint64(h)).astype(np.int64) & ((1 << (N - h)) - 1)
    b = (n & np.uint64((1 << h) - 1)).astype(np.int64)
    return np.where(ok, Ja[a] + Jb[b], -1).astype(np.int64)


def clt_bytes(N: int) -> int:
    """Eq. 21 (L177-L181): 8 bytes per block of 32 labels."""
    return 8 * (((1 << N) + 31) // 32)


def nnz_formula(N: int, N_up: int, n_bonds: int) -> int:
    """Eq. 10 (L78-L82) at s = 1/2: N_nz = D_M(N) + 2 N_B D(N-2 sites, N_up-1 ups)
    (for s = 1/2 the a,b sum has the single term a = -1/2, b = +1/2)."""
    off = math.comb(N - 2, N_up - 1) if 1 <= N_up <= N - 1 else 0
    return math.comb(N, N_up) + 2 * n_bonds * off


# --------------------------------------------------------------------------------------
# O2  Hamiltonian (Eqs. 1, 12-14 at s = 1/2; L27-L32, L105-L115)
# --------------------------------------------------------------------------------------


def ladder_coeffs(J: float, m_i: float, m_j: float, s: float = 0.5):
    """Eqs. 13-14 (L111-L115) verbatim.  c+ belongs to the source state with
    (m_i - 1, m_j + 1), c- to (m_i + 1, m_j - 1); a coefficient whose source quantum
    numbers leave [-s, s] is zero (the square root's argument vanishes)."""
    def rt(x):
        return math.sqrt(max(x, 0.0))
    cp = 0.5 * J * rt(s * (s + 1) - m_i * (m_i - 1)) * rt(s * (s + 1) - m_j * (m_j + 1))
    cm = 0.5 * J * rt(s * (s + 1) - m_i * (m_i + 1)) * rt(s * (s + 1) - m_j * (m_j - 1))
    return cp, cm


def diagonal(basis, N, bond_i, bond_j, J, h, N_up) -> np.ndarray:
    """First term of Eq. 12 (L107): sum_b J_b m_i m_j, m = +-1/2, plus the constant
    Zeeman shift -h M_z of reading 5."""
    d = np.zeros(basis.shape[0], dtype=np.float64)
    for b in range(len(J)):
        si = ((basis >> np.uint64(int(bond_i[b]))) & np.uint64(1)).astype(np.float64) - 0.5
        sj = ((basis >> np.uint64(int(bond_j[b]))) & np.uint64(1)).astype(np.float64) - 0.5
        d += J[b] * si * sj
    return d - h * (N_up - N / 2.0)


def apply_H(basis, N, bond_i, bond_j, J, h, N_up, v) -> np.ndarray:
    """y = H v in the sector, row-wise gather (Eq. 12): y[t] = diag(n_t) v[t] +
    sum over bonds with antiparallel spins of (J_b/2) v[index(n_t with both spins
    flipped)].  (At s = 1/2 exactly one of c+, c- equals J/2 on an antiparallel bond and
    both vanish otherwise: reading 6, checked in tests against `ladder_coeffs`.)"""
    v = np.asarray(v, dtype=np.float64)
    y = diagonal(basis, N, bond_i, bond_j, J, h, N_up) * v
    for b in range(len(J)):
        i, j = int(bond_i[b]), int(bond_j[b])
        bi = (basis >> np.uint64(i)) & np.uint64(1)
        bj = (basis >> np.uint64(j)) & np.uint64(1)
        anti = bi != bj
        src = basis[anti] ^ np.uint64((1 << i) | (1 << j))
        idx = index_of_sorted(basis, src)
        assert (idx >= 0).all()            # M_z is conserved (L165)
        y[anti] += 0.5 * J[b] * v[idx]
    return y


def apply_H_sampled_rows(N, bond_i, bond_j, J, h, N_up, rows, v_of) -> np.ndarray:
    """Rows `rows` of y = H v (the same Eq. 12) for a sector too large to enumerate (config 5:
    D = 2.33e9): the label of row t comes from the inverse map (L136), the index of every flipped label from
    Algorithm 1 (L138-L144), and the input vector is a callable `v_of(indices) -> values` (e.g. the counter-based
    start vector of DESIGN.md section 4, which has random access).  No basis array, no search.
    Pinned in tests/test_oracle_hamiltonian.py against `apply_H` on every row of small sectors."""
    rows = np.asarray(rows, dtype=np.int64)
    _, Dc = cr_tables(N)
    lab = alg1_unrank_vec(rows.astype(np.uint64), N, N_up, Dc)
    y = diagonal(lab, N, bond_i, bond_j, J, h, N_up) * np.asarray(v_of(rows), dtype=np.float64)
    for b in range(len(J)):
        i, j = int(bond_i[b]), int(bond_j[b])
        anti = ((lab >> np.uint64(i)) & np.uint64(1)) != ((lab >> np.uint64(j)) & np.uint64(1))
        src = alg1_rank_vec(lab[anti] ^ np.uint64((1 << i) | (1 << j)), N, N_up, Dc)
        y[anti] += 0.5 * J[b] * np.asarray(v_of(src), dtype=np.float64)
    return y


def neighbor_indices(basis, bond_i, bond_j, rows) -> np.ndarray:
    """Source index per (row, bond): index of the flipped label, -1 where the bond's spins
    are parallel (no off-diagonal element).  Used for the bit-exact neighbour check."""
    rows = np.asarray(rows, dtype=np.int64)
    out = np.full((rows.shape[0], len(bond_i)), -1, dtype=np.int64)
    lab = basis[rows]
    for b in range(len(bond_i)):
        i, j = int(bond_i[b]), int(bond_j[b])
        anti = ((lab >> np.uint64(i)) & np.uint64(1)) != ((lab >> np.uint64(j)) & np.uint64(1))
        out[anti, b] = index_of_sorted(basis, lab[anti] ^ np.uint64((1 << i) | (1 << j)))
    return out


def dense_H(N, bond_i, bond_j, J, h, N_up) -> np.ndarray:
    """Explicit sector matrix, element by element from O2."""
    basis = sector_basis(N, N_up)
    D = basis.shape[0]
    H = np.zeros((D, D), dtype=np.float64)
    H[np.arange(D), np.arange(D)] = diagonal(basis, N, bond_i, bond_j, J, h, N_up)
    for b in range(len(J)):
        i, j = int(bond_i[b]), int(bond_j[b])
        anti = ((basis >> np.uint64(i)) & np.uint64(1)) != ((basis >> np.uint64(j)) & np.uint64(1))
        rows = np.nonzero(anti)[0]
        cols = index_of_sorted(basis, basis[rows] ^ np.uint64((1 << i) | (1 << j)))
        np.add.at(H, (rows, cols), 0.5 * J[b])
    return H


def full_space_H_kron(N, bond_i, bond_j, J, h=0.0) -> np.ndarray:
    """Independent construction used only as a pin: H = sum_b J_b [Sz Sz + (S+S- + S-S+)/2]
    - h sum_i Sz_i on the full 2^N space from Kronecker products of 2x2 spin matrices
    (Eq. 1).  Site k is bit k of the label, so site 0 is the fastest index."""
    sz = np.array([[-0.5, 0.0], [0.0, 0.5]])      # basis order: bit 0 (down), bit 1 (up)
    sp = np.array([[0.0, 0.0], [1.0, 0.0]])       # S+ |down> = |up>
    sm = sp.T
    I2 = np.eye(2)

    def op(site_ops):
        M = np.array([[1.0]])
        for k in range(N - 1, -1, -1):            # leftmost factor = most significant bit
            M = np.kron(M, site_ops.get(k, I2))
        return M

    dim = 1 << N
    H = np.zeros((dim, dim))
    for b in range(len(J)):
        i, j = int(bond_i[b]), int(bond_j[b])
        H += J[b] * (op({i: sz, j: sz}) + 0.5 * (op({i: sp, j: sm}) + op({i: sm, j: sp})))
    if h != 0.0:
        for k in range(N):
            H -= h * op({k: sz})
    return H


# --------------------------------------------------------------------------------------
# Start vectors: the counter-based Gaussian generator specified in DESIGN.md section 4
# (readings 12-14).  Both sides implement this text independently.
# --------------------------------------------------------------------------------------

_GOLD = np.uint64(0x9E3779B97F4A7C15)


def _mix64(x):
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = (x ^ (x >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        x = (x ^ (x >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return x ^ (x >> np.uint64(31))


def chain_key(seed: int, N_up: int, r: int) -> np.uint64:
    with np.errstate(over="ignore"):
        k = _mix64(np.uint64(seed & ((1 << 64) - 1)))
        k = _mix64(k + _GOLD * np.uint64(N_up + 1))
        k = _mix64(k + _GOLD * np.uint64(r + 1))
    return k


def gaussian_elements(seed: int, N_up: int, r: int, t) -> np.ndarray:
    """Unnormalised N(0,1) element(s) t of start vector r in sector N_up: Box-Muller,
    g = sqrt(-2 ln u1) cos(2 pi u2), u1 = (a>>11 + 1) 2^-53 in (0,1], u2 = (b>>11) 2^-53,
    a = mix(key + GOLD (2t+1)), b = mix(key + GOLD (2t+2))."""
    t = np.asarray(t, dtype=np.uint64)
    key = chain_key(seed, N_up, r)
    with np.errstate(over="ignore"):
        a = _mix64(key + _GOLD * (np.uint64(2) * t + np.uint64(1)))
        b = _mix64(key + _GOLD * (np.uint64(2) * t + np.uint64(2)))
    u1 = ((a >> np.uint64(11)).astype(np.float64) + 1.0) * 2.0 ** -53
    u2 = (b >> np.uint64(11)).astype(np.float64) * 2.0 ** -53
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(6.283185307179586 * u2)


def start_vector(seed: int, N_up: int, r: int, D: int, chunk: int = 1 << 22) -> np.ndarray:
    """Normalised random start vector |r> (L34; Gaussian per BASELINE): g / ||g||_2."""
    g = np.empty(D, dtype=np.float64)
    for lo in range(0, D, chunk):
        hi = min(D, lo + chunk)
        g[lo:hi] = gaussian_elements(seed, N_up, r, np.arange(lo, hi, dtype=np.uint64))
    return g / math.sqrt(float(np.dot(g, g)))


def start_vector_norm(seed: int, N_up: int, r: int, D: int, chunk: int = 1 << 22) -> float:
    s = 0.0
    for lo in range(0, D, chunk):
        g = gaussian_elements(seed, N_up, r, np.arange(lo, min(D, lo + chunk), dtype=np.uint64))
        s += float(np.dot(g, g))
    return math.sqrt(s)


# --------------------------------------------------------------------------------------
# O3/O4  Lanczos without re-orthogonalisation and Ritz weights (L45)
# --------------------------------------------------------------------------------------


def lanczos(matvec, q1, n_steps: int, tol: float = 1e-12):
    """q_0 = 0, beta_0 = 0; for j = 1..m: w = H q_j - beta_{j-1} q_{j-1};
    alpha_j = <q_j, w>; w <- w - alpha_j q_j; beta_j = ||w||; q_{j+1} = w / beta_j
    (reading 7).  m = min(n_steps, D) (reading 9).  Breakdown (reading 10): stop with
    m_eff = j when beta_j <= tol * max_k(|alpha_k|, beta_k).  Returns alpha[0:m_eff],
    beta[0:m_eff-1]."""
    q = np.asarray(q1, dtype=np.float64).copy()
    D = q.shape[0]
    m = min(n_steps, D)
    q_prev = np.zeros(D)
    beta_prev = 0.0
    alpha, beta = [], []
    scale = 0.0
    for j in range(1, m + 1):
        w = matvec(q) - beta_prev * q_prev
        a = float(np.dot(q, w))
        alpha.append(a)
        if j == m:
            break
        w = w - a * q
        bnorm = math.sqrt(float(np.dot(w, w)))
        scale = max(scale, abs(a), bnorm)
        if bnorm <= tol * scale:
            break
        beta.append(bnorm)
        q_prev, q, beta_prev = q, w / bnorm, bnorm
    return np.array(alpha), np.array(beta)


def ritz(alpha, beta):
    """Eigenpairs (theta_k, s_k) of the tridiagonal T; weights w_k = |s_{k,1}|^2 (L45)."""
    m = len(alpha)
    T = np.diag(np.asarray(alpha, dtype=np.float64))
    if m > 1:
        T += np.diag(np.asarray(beta[: m - 1], dtype=np.float64), 1)
        T += np.diag(np.asarray(beta[: m - 1], dtype=np.float64), -1)
    theta, S = np.linalg.eigh(T)
    return theta, S[0, :] ** 2


# --------------------------------------------------------------------------------------
# O5  FTLM thermodynamics (Eqs. 4-9)
# --------------------------------------------------------------------------------------


def thermo(sectors, T_grid, g: float = 2.0):
    """sectors: list of dicts {dim, Mz, mult, chains: [(theta, w), ...]} (mult = 2 for
    M_z > 0: reading 15).  Z = sum_sec mult (D/R) sum_r sum_k w e^{-theta/T} (Eq. 7);
    <H^p> by Eq. 8; E = <H>; C = (<H^2> - <H>^2)/T^2 (L67); chi = g^2 sum M_z^2 Z_M /
    (T sum Z_M) (Eq. 9).  Exponentials are taken relative to E_ref = min theta
    (reading 17); returns dict(E_ref, Zs = Z e^{E_ref/T}, E, C, chi)."""
    T_grid = np.asarray(T_grid, dtype=np.float64)
    E_ref = min(float(np.min(th)) for s in sectors for th, _ in s["chains"])
    Z = np.zeros_like(T_grid)
    H1 = np.zeros_like(T_grid)
    H2 = np.zeros_like(T_grid)
    M2 = np.zeros_like(T_grid)
    for s in sectors:
        R = len(s["chains"])
        pref = s["mult"] * s["dim"] / R
        Zs = np.zeros_like(T_grid)
        for th, w in s["chains"]:
            e = np.exp(-(th[None, :] - E_ref) / T_grid[:, None]) * w[None, :]
            Zs += pref * e.sum(axis=1)
            H1 += pref * (e * th[None, :]).sum(axis=1)
            H2 += pref * (e * th[None, :] ** 2).sum(axis=1)
        Z += Zs
        M2 += s["Mz"] ** 2 * Zs
    E = H1 / Z
    C = (H2 / Z - E ** 2) / T_grid ** 2
    chi = g ** 2 * M2 / (T_grid * Z)
    return dict(E_ref=E_ref, Zs=Z, E=E, C=C, chi=chi)


def exact_thermo(spectra, T_grid, g: float = 2.0):
    """O6: exact Z, E, C, chi from complete sector spectra.  spectra: list of
    (Mz, mult, eigenvalues)."""
    secs = [dict(dim=len(ev), Mz=Mz, mult=mult,
                 chains=[(np.asarray(ev, dtype=np.float64), np.full(len(ev), 1.0 / len(ev)))])
            for Mz, mult, ev in spectra]
    return thermo(secs, T_grid, g)


def ftlm_run(N, bond_i, bond_j, J, h, N_up_list, R, n_steps, seed, T_grid, tol=1e-12,
             cast=None):
    """Whole FTLM of config-1 style (L32, L45, L61-L76): for each sector M_z >= 0, R seeded
    Gaussian starts, Lanczos, Ritz pairs; then `thermo`.  `cast` (optional) rounds each start
    vector through another dtype before use (FP32-mode comparisons start from the same
    FP32-rounded vector, reading 13)."""
    secs = []
    coeffs = {}
    for N_up in N_up_list:
        basis = sector_basis(N, N_up)
        D = basis.shape[0]
        mv = lambda x, _b=basis, _n=N_up: apply_H(_b, N, bond_i, bond_j, J, h, _n, x)
        chains = []
        for r in range(R):
            q1 = start_vector(seed, N_up, r, D)
            if cast is not None:
                q1 = q1.astype(cast).astype(np.float64)
            a, b = lanczos(mv, q1, n_steps, tol)
            coeffs[(N_up, r)] = (a, b)
            chains.append(ritz(a, b))
        Mz = N_up - N / 2.0
        secs.append(dict(dim=D, Mz=Mz, mult=(1 if Mz == 0 else 2), chains=chains))
    return thermo(secs, T_grid), secs, coeffs


# --------------------------------------------------------------------------------------
# Diagnostics: ghost flags, cluster weights, stochastic error estimates
# --------------------------------------------------------------------------------------

U_FP32 = 2.0 ** -24


def ghost_diagnostic(alpha, beta, C_tau: float = 1.0):
    """Cullum-Willoughby test as the paper states it (L258-L262, Eq. 25): T^(1) = T without its first row and
    column, l_k = min_j |theta_k - theta^(1)_j|, ghost iff l_k < tau, tau = C_tau u_FP32 W_T with
    W_T = theta_max - theta_min (one tolerance for both precisions).  Clusters (L270): theta_k and theta_l belong
    together whenever |theta_k - theta_l| <= tau (chains of such neighbours join); the meaningful weight of a
    cluster is the sum of its members' weights.  Also the cumulative spectral weight F(theta_k) of Eq. 23 (L248).
    Returns dict(theta, weight, ell, tau, ghost (bool), cluster (id per k, ascending), cluster_weight (per k:
    the total weight of k's cluster), F)."""
    theta, w = ritz(alpha, beta)
    m = len(theta)
    if m > 1:
        theta1, _ = ritz(np.asarray(alpha)[1:], np.asarray(beta)[1:m - 1] if m > 2 else [])
        ell = np.min(np.abs(theta[:, None] - theta1[None, :]), axis=1)
    else:
        ell = np.full(m, np.inf)
    tau = C_tau * U_FP32 * (theta[-1] - theta[0]) if m else 0.0
    ghost = ell < tau
    cluster = np.zeros(m, dtype=np.int64)
    for k in range(1, m):
        cluster[k] = cluster[k - 1] + (0 if theta[k] - theta[k - 1] <= tau else 1)
    cw = np.array([w[cluster == cluster[k]].sum() for k in range(m)])
    return dict(theta=theta, weight=w, ell=ell, tau=tau, ghost=ghost, cluster=cluster, cluster_weight=cw, F=np.cumsum(w))


def sigma_emp(samples):
    """Eq. 22 (L225-L228): samples[s][i] = FTLM estimate of the observable at seed set s and temperature i;
    sigma_emp = sqrt((1/N_s) sum_s (O_s - mean)^2) (population form, as printed).  Returns (mean, sigma)."""
    a = np.asarray(samples, dtype=np.float64)
    mean = a.mean(axis=0)
    return mean, np.sqrt(((a - mean[None, :]) ** 2).mean(axis=0))


def sigma_theo(O, Z_eff):
    """L230: sigma_theo = O / sqrt(Z_eff), Z_eff = Tr exp(-(H - E_0)/T) (here: the FTLM estimate Zs of `thermo`,
    whose reference energy is the lowest Ritz value)."""
    return np.abs(np.asarray(O, dtype=np.float64)) / np.sqrt(np.asarray(Z_eff, dtype=np.float64))
