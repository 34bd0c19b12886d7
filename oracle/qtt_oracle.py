"""CPU ORACLE (TEST INFRASTRUCTURE, NOT PRODUCT CODE) for the per-time-step MPS
algebra of the quantics-tensor-train (QTT/MPS) 2D Navier-Stokes solver of
arxiv 2406.17823 (Hoelscher et al.), written from /root/reference/PAPER.md.

Plain, slow, obviously-correct NumPy fp64.  LAPACK ``qr``/``svd`` and
``einsum``/``matmul`` are the only library steps.  It shares no code with the
CUDA path (paper_2406_17823_b200/) and neither imports the other.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.

Data model (Sec. II.B, Eq. 3-4): a field F[x][y] on an N x N
grid, N = 2**n, becomes an n-site MPS; site k = 1..n carries
omega_k = 2*x_bit_k + y_bit_k with bit 1 the MOST significant (PAPER.md:59-67
Eq. 3; "alpha_{m+1} connected to the tensor of the less
significant bits").  An MPS is a Python list of n arrays ``core[k]`` of shape
(r_{k-1}, 4, r_k), r_0 = r_n = 1.  An MPO is a list of n arrays of shape
(D_{k-1}, 4, 4, D_k) indexed [alpha_{k-1}][omega (output)][omega' (input)][alpha_k],
D_0 = D_n = 1 (boundary vectors L, R of PAPER.md:90-98 Eq. 7 folded into the
end cores).

Functions and the passage each follows (DESIGN.md "Readings" lists every point
where the paper is silent/garbled and the reading taken):

  O1  encode / decode           PAPER.md:59-67  Eq. 3 (quantics bit interleave)
  O2  from_dense                PAPER.md:67-72  Eq. 4; R->L TT-SVD (ref. [15])
  O3  apply_mpo                 PAPER.md:85     "act on them by contracting the respective indices"
  O4  hadamard                  PAPER.md:100-105 Eq. 8, Fig. 2(a) (bond chi^2)
  O5  lincomb / axpy            PAPER.md:126-130 Eq. 11 (sum of RK4 pieces)
  O6  round                     PAPER.md:130 ("compression ... repeated SVDs"), ref. [15];
                                eps semantics PAPER.md:238 Eq. 16
  O7  round_product (zip-up)    PAPER.md:105 ("needs to be compressed down to chi again");
                                the chi^2 product is never formed
  O8  rhs                       PAPER.md:49-53 Eq. 2 without pressure (Burgers form)
  O9  rk4_step                  PAPER.md:124-128 Eq. 11
  O10 mpo_d1 / mpo_d2 / mpo_laplacian   PAPER.md:391-424 App. A, Eq. A1-A3, Table II
      mpo_stencil (any order)   PAPER.md:98, same construction
  O11 fidelity, chi_eps         PAPER.md:160 Eq. 12; Eq. 16-17 (diagnostics)
      tke_spectrum              PAPER.md:173-184 Eq. 13-15
  O12 variational_cost / variational_stage   PAPER.md:107-132 Sec. II.C; 437-452 Eq. B3-B6; 522-544 Eq. B20-B24
  O13 sketch_signs / sketch_mixers / sketch_probes / sketch_factor / sketch_applies, round_product(sketch_seed=)
                                PAPER.md:318 ("cheaper product compression"; reading 25: randomised range finder)

  P1-P4 (oracle/qtt_oracle_3d.py) the 3D encoding with physical dimension 8: encode3, from_dense3, mpo_stencil3 / mpo_d3 /
                                mpo_laplacian3, rhs3 / rk4_step3 (reading 26); O3-O7 here read the
                                physical dimension off the core shapes and serve both encodings

Pins (tests/test_oracle_*.py, ``-m "not gpu"``): dense brute force on 2^4..2^6
grids, Table II golden entries (tests/golden/), circulant stencil of Eq. 6,
analytic finite-difference of sin/cos, bond-2 closed forms, the root-sum-square
truncation identity, norm preservation, dense TT-SVD, dense RK4 of the same
stencils.

Parity-pin status: O1-O11 pinned.  O7 with a working bond that really truncates is algorithm-defined
(reading 8), and each of its steps is pinned in tests/test_oracle_zipup_pins.py: per site Q^T Q = I,
R' = Q^T T, ||T - Q R'||_F = the tail of an independent svdvals(T) beyond keep = min(chi_work, rows, cols)
(Eckart-Young), T_l = (Phi_{<l}^T (x) I_4) X_l with X_l from the explicit hadamard() cores, a planted spectrum
with a gap at chi_work, and the projected dense product as the state handed to the R->L sweep; the eps rank
rule by hand-computed tails, brute-force minimality and a case where the 1/sqrt(n-1) split decides the rank.
O12 (variational stage) is pinned in tests/test_oracle_variational.py by the dense normal equations of Theta,
finite-difference stationarity at truncating bonds and the dense operator product.
O13 (sketched zip-up) is pinned in tests/test_oracle_sketch.py by a big-integer restatement of the generator, the dense
probe train, projector algebra, the range-finder bound against independent SVDs of the matrix and of the true unfolding,
gauge invariance and the dense elementwise product.
"""
from __future__ import annotations

import math
import numpy as np

D_PHYS = 4  # physical dimension d = 2^k for a k-dimensional grid, k = 2


# --------------------------------------------------------------------------- O1
def encode(F: np.ndarray) -> np.ndarray:
    """Dense F[x][y] (N x N) -> tensor U[w_1]...[w_n], w_k = 2*x_bit_k + y_bit_k,
    bit 1 most significant (Eq. 3)."""
    N = F.shape[0]
    n = int(round(math.log2(N)))
    assert F.shape == (N, N) and (1 << n) == N
    T = np.asarray(F, dtype=np.float64).reshape((2,) * n + (2,) * n)  # x bits msb..lsb, y bits msb..lsb
    perm = []
    for k in range(n):
        perm += [k, n + k]
    return T.transpose(perm).reshape((D_PHYS,) * n)


def decode(U: np.ndarray) -> np.ndarray:
    """Inverse of :func:`encode`."""
    n = U.ndim
    N = 1 << n
    T = U.reshape((2, 2) * n)  # x1 y1 x2 y2 ...
    perm = [2 * k for k in range(n)] + [2 * k + 1 for k in range(n)]
    return T.transpose(perm).reshape(N, N)


# ---------------------------------------------------------------- rank rule (O6)
def _rank_rule(s: np.ndarray, chi_max: int, delta) -> int:
    """Kept rank r' for singular values s (descending).

    eps = 0 (delta is None): r' = min(chi_max, len(s))  (static shapes, no thresholding).
    eps > 0: smallest r with sqrt(sum_{i>r} s_i^2) <= delta, then
    r' <- max(1, min(r, chi_max)).  (reading 6; eps is the total
    relative error of PAPER.md:238 Eq. 16, split evenly over the n-1 bonds.)
    """
    m = len(s)
    if delta is None:
        return max(1, min(int(chi_max), m))
    tail = np.sqrt(np.cumsum((s[::-1]) ** 2))[::-1]  # tail[r] = sqrt(sum_{i>=r} s_i^2)
    r = m
    for cand in range(m + 1):
        t = tail[cand] if cand < m else 0.0
        if t <= delta:
            r = cand
            break
    return max(1, min(r, int(chi_max), m))


# --------------------------------------------------------------------------- O2
def from_dense(F: np.ndarray, chi_max: int = 1 << 30, eps: float = 0.0):
    """TT-SVD proceeding right-to-left (Eq. 4; reading 9):
    for k = n..2, SVD the 4^{k-1} x (4 r_k) unfolding, keep r by the rank rule,
    core_k = V^T, carry U S; core_1 = carry."""
    U = encode(F)
    n = U.ndim
    nrm = float(np.linalg.norm(U))
    delta = eps * nrm / math.sqrt(max(n - 1, 1)) if eps > 0 else None
    cores = [None] * n
    carry = U.reshape(-1, 1)  # (4^n) x r_n, r_n = 1
    r = 1
    for k in range(n, 1, -1):
        M = carry.reshape(D_PHYS ** (k - 1), D_PHYS * r)
        Um, s, Vt = np.linalg.svd(M, full_matrices=False)
        rk = _rank_rule(s, chi_max, delta)
        cores[k - 1] = Vt[:rk].reshape(rk, D_PHYS, r)
        carry = Um[:, :rk] * s[:rk]
        r = rk
    cores[0] = carry.reshape(1, D_PHYS, r)
    return cores


def to_tensor(cores) -> np.ndarray:
    """Contract an MPS to the full tensor U[w_1..w_n] (Eq. 4)."""
    T = cores[0].reshape(cores[0].shape[1], -1)
    for c in cores[1:]:
        r0, d, r1 = c.shape
        T = (T @ c.reshape(r0, d * r1)).reshape(-1, r1)
    return T.reshape((cores[0].shape[1],) * len(cores))


def to_dense(cores) -> np.ndarray:
    """MPS -> dense F[x][y]."""
    return decode(to_tensor(cores))


def bonds(cores):
    return [1] + [c.shape[2] for c in cores]


# --------------------------------------------------------------------------- O3
def apply_mpo(W, A):
    """B[(alpha,a), w, (beta,b)] = sum_{w'} W[alpha, w, w', beta] * A[a, w', b]
    (MPO bond index major).  Exact, bond D*chi."""
    out = []
    for Wk, Ak in zip(W, A):
        Dl, d, _, Dr = Wk.shape
        a, _, b = Ak.shape
        B = np.einsum("xopy,apb->xaoyb", Wk, Ak)
        out.append(B.reshape(Dl * a, d, Dr * b))
    return out


# --------------------------------------------------------------------------- O4
def hadamard(A, B):
    """C[(a,b), w, (a',b')] = A[a,w,a'] * B[b,w,b'] (Eq. 8:
    |u_i> (.) as an MPO with rank-3 Kronecker deltas; bond chi_a*chi_b)."""
    out = []
    for Ak, Bk in zip(A, B):
        a, d, a2 = Ak.shape
        b, _, b2 = Bk.shape
        C = np.einsum("awc,bwd->abwcd", Ak, Bk)
        out.append(C.reshape(a * b, d, a2 * b2))
    return out


# --------------------------------------------------------------------------- O5
def lincomb(terms):
    """sum_j alpha_j |X_j> as an MPS by direct sum: first core
    [alpha_1 X_1 | alpha_2 X_2 | ...], middle cores block-diagonal, last cores
    stacked.  ``terms`` = [(alpha, cores), ...].  The scalar sits on the first core."""
    n = len(terms[0][1])
    k = len(terms)
    out = []
    for site in range(n):
        cs = [t[1][site] for t in terms]
        if site == 0:
            out.append(np.concatenate([t[0] * c for t, c in zip(terms, cs)], axis=2))
        elif site == n - 1:
            out.append(np.concatenate(cs, axis=0))
        else:
            rl = sum(c.shape[0] for c in cs)
            rr = sum(c.shape[2] for c in cs)
            blk = np.zeros((rl, cs[0].shape[1], rr))
            i = j = 0
            for c in cs:
                blk[i : i + c.shape[0], :, j : j + c.shape[2]] = c
                i += c.shape[0]
                j += c.shape[2]
            out.append(blk)
    assert k >= 1
    return out


def axpy(alpha, X, Y):
    """alpha*X + Y (exact)."""
    return lincomb([(alpha, X), (1.0, Y)])


# --------------------------------------------------------------------------- O6
def _sweep_lr(cores):
    """(i) L->R: thin QR of each left unfolding, R into the next core."""
    cores = [c.copy() for c in cores]
    n = len(cores)
    for k in range(n - 1):
        r0, d, r1 = cores[k].shape
        Q, R = np.linalg.qr(cores[k].reshape(r0 * d, r1))  # reduced
        rq = Q.shape[1]
        cores[k] = Q.reshape(r0, d, rq)
        nr0, _, nr1 = cores[k + 1].shape
        cores[k + 1] = (R @ cores[k + 1].reshape(nr0, d * nr1)).reshape(rq, d, nr1)
    return cores


def _sweep_rl(cores, chi_max, eps, info=None):
    """(ii) R->L for k = n..2: SVD of the right unfolding; rank rule; core_k <- V^T[:r'],
    left neighbour <- left * (U[:, :r'] S[:r']).  ``cores`` must be left-orthogonal
    up to the last site, so ||A||_F = ||last core||."""
    n = len(cores)
    nrm = float(np.linalg.norm(cores[-1]))
    delta = eps * nrm / math.sqrt(max(n - 1, 1)) if eps > 0 else None
    if info is not None:
        info["norm"] = nrm
        info["singular_values"] = [None] * (n + 1)
        info["discarded"] = [0.0] * (n + 1)
    for k in range(n - 1, 0, -1):
        r0, d, r1 = cores[k].shape
        U, s, Vt = np.linalg.svd(cores[k].reshape(r0, d * r1), full_matrices=False)
        rk = _rank_rule(s, chi_max, delta)
        cores[k] = Vt[:rk].reshape(rk, d, r1)
        US = U[:, :rk] * s[:rk]
        p0, _, _ = cores[k - 1].shape
        cores[k - 1] = (cores[k - 1].reshape(p0 * d, r0) @ US).reshape(p0, d, rk)
        if info is not None:
            info["singular_values"][k] = s.copy()
            info["discarded"][k] = float(np.sqrt(np.sum(s[rk:] ** 2)))
    return cores


def round_mps(cores, chi_max: int = 1 << 30, eps: float = 0.0, info=None):
    """TT-rounding (ref. [15] of the paper).  Never normalises; a zero
    MPS stays zero.  Output is right-canonical (norm on site 1)."""
    return _sweep_rl(_sweep_lr(cores), chi_max, eps, info)


# --------------------------------------------------------------------------- O7
_M64 = (1 << 64) - 1


def sketch_signs(seed: int, site: int, rows: int, cols: int) -> np.ndarray:
    """Random signs Omega[c, t] in {+1, -1} of the sketched zip-up (reading 25), a counter-based generator both
    sides implement: z = seed * 0x9E3779B97F4A7C15 + site * 0xD1B54A32D192ED03 + c * 2^20 + t (mod 2^64), mixed by the
    splitmix64 finaliser z ^= z >> 30; z *= 0xBF58476D1CE4E5B9; z ^= z >> 27; z *= 0x94D049BB133111EB; z ^= z >> 31;
    Omega = -1 if the top bit of z is set, else +1.  (cols < 2^20.)  The zip-up uses it with rows = 4 P (sketch_mixers)."""
    base = (int(seed) * 0x9E3779B97F4A7C15 + int(site) * 0xD1B54A32D192ED03) & _M64
    c = np.arange(rows, dtype=np.uint64)[:, None]
    t = np.arange(cols, dtype=np.uint64)[None, :]
    with np.errstate(over="ignore"):
        z = np.uint64(base) + (c << np.uint64(20)) + t
        z ^= z >> np.uint64(30)
        z *= np.uint64(0xBF58476D1CE4E5B9)
        z ^= z >> np.uint64(27)
        z *= np.uint64(0x94D049BB133111EB)
        z ^= z >> np.uint64(31)
    return np.where((z >> np.uint64(63)) == 1, -1.0, 1.0)


def sketch_mixers(seed: int, site: int, n_probes: int) -> np.ndarray:
    """G[w][u][t] = sketch_signs(seed, site, 4 P, P)[w P + u, t] / sqrt(P), P = n_probes: site `site`'s core of the random
    tensor train the probes are (physical index w, bonds u -> t)."""
    P = int(n_probes)
    return sketch_signs(seed, site, D_PHYS * P, P).reshape(D_PHYS, P, P) * (1.0 / math.sqrt(P))


def sketch_probes(A, B, n_probes: int, seed: int):
    """Structured probes of the sketched zip-up (reading 25): a random tensor train over the PHYSICAL indices with bond P =
    n_probes and sign cores G_k (sketch_mixers; sites k counted from 0; the open bond t at the left end numbers the probes),
        Omega[w_l .. w_{n-1}; t] = sum_{u's} G_l[w_l][u_{l+1}, t] G_{l+1}[w_{l+1}][u_{l+2}, u_{l+1}] ... G_{n-1}[w_{n-1}][u_n, u_{n-1}],
    closed by the all-ones vector at u_n.  Contracted through the product's own site tensors from the right they give, for
    every bond l,
        S_l[a, b, t] = sum_{w, u} G_l[w][u, t] sum_{a', b'} A_l[a, w, a'] B_l[b, w, b'] S_{l+1}[a', b', u],     S_n = 1,
    i.e. the probes as seen from the bond (a, b) left of site l.  Because they live on the physical indices, T S is the
    same whatever gauge the bonds of A and B are in -- a random matrix on the bond indices themselves would not be
    (measured: two gauges of the same operand gave results 10 % apart).  Probes with bond 1 (one rank-one tensor of sign
    vectors per probe) are cheaper still but fail too often: over 12 seeds their worst range-finder error was 12 .. 1000 x the
    optimal rank-P/2 tail of the unfolding, against 0.08 .. 1.07 x for the bond-P train (randomised TT rounding in the
    literature uses such trains for the same reason).  Returns [S_0, ..., S_n]."""
    n = len(A)
    S = [None] * (n + 1)
    S[n] = np.ones((1, 1, n_probes))
    for l in range(n - 1, -1, -1):
        G = sketch_mixers(seed, l, n_probes)
        a, b = A[l].shape[0], B[l].shape[0]
        S[l] = np.zeros((a, b, n_probes))
        for w in range(D_PHYS):  # the formula above, one physical index at a time (plain matrix products)
            X = np.tensordot(A[l][:, w, :], S[l + 1], axes=([1], [0]))  # [a, b', u]
            Z = X @ G[w]  # [a, b', t]
            S[l] += np.tensordot(Z, B[l][:, w, :], axes=([1], [1])).transpose(0, 2, 1)  # [a, t, b] -> [a, b, t]
    return S


def sketch_factor(T: np.ndarray, Sl: np.ndarray):
    """The truncating step of the sketched zip-up: Q = an orthonormal basis of the numerical range of Y = T S (left singular
    vectors of Y with sigma_i > 8 eps ||Y||_F; the columns beyond that rank are ZERO, so the bond keeps its size), S the
    probes seen from the right bond of this site as a (columns of T) x (probes) matrix, and R' = Q^T T: Q R' is the projection
    of T on the sketched range (randomised range finder; SURVEY.md section 8f next-4 "cheaper product compression",
    PAPER.md:318).  The rank cut makes the step a function of range(Y) alone: when Y is numerically rank deficient (smooth
    fields; coinciding probes) a plain QR would fill up with directions made of rounding noise."""
    Y = T @ Sl
    U, sv, _ = np.linalg.svd(Y, full_matrices=False)
    rank = int(np.sum(sv > 8.0 * np.finfo(np.float64).eps * np.linalg.norm(Y)))
    Q = np.zeros_like(U)
    Q[:, :rank] = U[:, :rank]
    return Q, Q.T @ T


def sketch_applies(n: int, l: int, m: int, k: int, chi_work: int) -> bool:
    """The sketch replaces the truncated SVD at zip-up site l (0-based) where that SVD really truncates (chi_work < min(m, k))
    and the c = 4^(n-1-l) physical configurations to the right of the site are either many, c >= 2 chi_work (the probes seen
    from bond l+1 span at most c dimensions: a random range finder wants them oversampled), or few, c <= chi_work: then the
    true unfolding has rank <= c <= chi_work, the probes span its whole range and the step loses nothing (DESIGN.md reading
    25).  In between (chi_work < c < 2 chi_work) the truncated SVD stays."""
    c = 4 ** (n - 1 - l)
    return chi_work < min(m, k) and (c >= 2 * chi_work or c <= chi_work)


def round_product(A, B, chi_max: int, eps: float = 0.0, chi_work: int | None = None, info=None, sketch_seed=None):
    """Fused Hadamard + round ("zip-up" with working bond chi_work; reading 8).

    carry R_0 = [1]; for l = 1..n-1:
        T = contract(R, A_l, B_l) as (4 r) x (a' b');
        if 4r <= min(a'b', chi_work):            Q = I,  R' = T
        elif a'b' < 4r and a'b' <= chi_work:     thin QR
        else:                                    truncated SVD keeping the chi_work largest
                                                 (Q = U, R' = S V^T)
        core_l = Q.
    Last site: core_n = contract(R, A_n, B_n).  Then step (ii) of O6 with (chi_max, eps).
    Default chi_work = 2*chi_max.  With chi_work >= every intermediate rank this IS
    round_mps(hadamard(A, B)).
    sketch_seed (an int): the cheaper compression of reading 25 -- wherever the line above takes a truncated SVD that
    really truncates (chi_work < min(4r, a'b')) and enough sites remain to the right (sketch_applies), take instead
    Q = orth(T S), R' = Q^T T with chi_work structured random probes (a sign tensor train) contracted through the remaining sites
    (sketch_probes, sketch_factor)."""
    if chi_work is None:
        chi_work = 2 * int(chi_max)
    n = len(A)
    R = np.ones((1, 1, 1))
    cores = []
    probes = None  # built at the first site that takes the sketch (a working bond that never truncates needs none)
    zip_log = []  # per site: the matrix T that was factorised, Q, R' and the branch taken (read by the pins only)
    for l in range(n - 1):
        T4 = np.einsum("rab,awc,bwd->rwcd", R, A[l], B[l], optimize=True)
        r, d, a2, b2 = T4.shape
        T = T4.reshape(r * d, a2 * b2)
        m, k = T.shape
        if m <= min(k, chi_work):
            Q = np.eye(m)
            Rn = T
            branch = "identity"
            s = None
        elif k < m and k <= chi_work:
            Q, Rn = np.linalg.qr(T)
            branch = "qr"
            s = None
        elif sketch_seed is not None and sketch_applies(n, l, m, k, chi_work):
            if probes is None:
                probes = sketch_probes(A, B, chi_work, sketch_seed)
            Q, Rn = sketch_factor(T, probes[l + 1].reshape(k, chi_work))
            branch = "sketch"
            s = None
        else:
            U, s, Vt = np.linalg.svd(T, full_matrices=False)
            keep = min(chi_work, len(s))
            Q = U[:, :keep]
            Rn = s[:keep, None] * Vt[:keep]
            branch = "svd"
        zip_log.append(dict(T=T, Q=Q, R=Rn, branch=branch, s=s))
        rn = Q.shape[1]
        cores.append(Q.reshape(r, d, rn))
        R = Rn.reshape(rn, a2, b2)
    T4 = np.einsum("rab,awc,bwd->rwcd", R, A[n - 1], B[n - 1], optimize=True)
    cores.append(T4.reshape(T4.shape[0], T4.shape[1], 1))
    if info is not None:
        info["zip"] = zip_log
        info["zip_cores"] = [c.copy() for c in cores]  # Q_1..Q_{n-1}, T_n: the state the R->L sweep starts from
    return _sweep_rl(cores, chi_max, eps, info)


# -------------------------------------------------------------------------- O10
# Table II of the paper, verbatim: (alpha_m, alpha_{m+1}, omega, omega') -> 1.
# C_{alpha_m alpha_{m+1}}^{omega omega'}.  omega = (x_m y_m)_2.
_TABLE_II = [
    (0, 0, 0, 0), (0, 0, 1, 1), (0, 0, 2, 2), (0, 0, 3, 3),   # alpha_{m+1} = 0: x +- 0
    (0, 1, 0, 2), (0, 1, 1, 3), (1, 1, 2, 0), (1, 1, 3, 1),   # alpha_{m+1} = 1: x + 1
    (2, 2, 0, 2), (2, 2, 1, 3), (0, 2, 2, 0), (0, 2, 3, 1),   # alpha_{m+1} = 2: x - 1
]


def _swap_bits(w: int) -> int:
    """Exchange the x and y bit of omega = (x y)_2."""
    return ((w & 1) << 1) | (w >> 1)


def shift_core(direction: int) -> np.ndarray:
    """Central core C[alpha_m][omega][omega'][alpha_{m+1}] of Table II, with omega the
    OUTPUT (row) index and omega' the index contracted with the MPS (reading 1:
    the literal text "output index omega'" yields -D, since D^T = -D).
    direction 1: shifts in x (Table II verbatim); direction 2: the same table with
    the roles of the x and y bit exchanged ("same logic")."""
    C = np.zeros((3, D_PHYS, D_PHYS, 3))
    for am, am1, w, wp in _TABLE_II:
        if direction == 2:
            w, wp = _swap_bits(w), _swap_bits(wp)
        C[am, w, wp, am1] = 1.0
    return C


def _fold_boundaries(core_list, L, R):
    out = [c.copy() for c in core_list]
    out[0] = np.einsum("x,xopy->opy", L, out[0])[None]
    out[-1] = np.einsum("xopy,y->xop", out[-1], R)[..., None]
    return out


def mpo_d1(n: int, dx: float):
    """Central-difference MPO D_1 (PAPER.md:395-404 Eq. A1-A3): L = (1,1,1) on the
    most-significant end, R = (0, 1, -1)/(2 dx) on the least-significant end."""
    C = shift_core(1)
    return _fold_boundaries([C] * n, np.ones(3), np.array([0.0, 1.0, -1.0]) / (2.0 * dx))


def mpo_d2(n: int, dx: float):
    """Same for the y direction."""
    C = shift_core(2)
    return _fold_boundaries([C] * n, np.ones(3), np.array([0.0, 1.0, -1.0]) / (2.0 * dx))


def mpo_laplacian(n: int, dx: float):
    """Compact 5-point Laplacian MPO, bond 5 (reading 3; not printed in the paper):
    channel 0 = identity, channels 1,2 = the alpha=1,2 entries of Table II for the
    x bit, channels 3,4 = the same for the y bit; L = (1,1,1,1,1),
    R = (-4, 1, 1, 1, 1)/dx^2."""
    C = np.zeros((5, D_PHYS, D_PHYS, 5))
    Cx, Cy = shift_core(1), shift_core(2)
    C[0, :, :, 0] = Cx[0, :, :, 0]  # identity channel
    for src, base in ((Cx, 0), (Cy, 2)):
        for a in (1, 2):
            C[0, :, :, base + a] = src[0, :, :, a]       # start a shift, no carry out
            C[base + a, :, :, base + a] = src[a, :, :, a]  # shift with carry out
    return _fold_boundaries([C] * n, np.ones(5), np.array([-4.0, 1.0, 1.0, 1.0, 1.0]) / dx**2)


def mpo_stencil(n: int, direction: int, coeffs):
    """General periodic finite-difference stencil along one direction as an MPO ("MPOs for finite-difference
    stencils of any order"):
        (O F)[x] = sum_{k=-K..K} coeffs[k + K] * F[x + k]      (x periodic, the other coordinate untouched),
    2K + 1 = len(coeffs).  Same construction as App. A: the bond carries the carry of the
    addition x + k, running from the least-significant site to the most-significant one.  Bond index
    alpha = carry + K, carry in [-K, K]; at a site with output bit b (of the shifted coordinate) and incoming carry c,
    the input bit is (b + c) mod 2 and the outgoing carry floor((b + c) / 2).  L = ones (periodic: the last carry is
    dropped), R[c + K] = coeffs[c + K] (the offset k enters as the initial carry).  Index order [alpha_m][w][w'][alpha_{m+1}],
    w = output (reading 1)."""
    coeffs = np.asarray(coeffs, dtype=np.float64)
    assert direction in (1, 2) and len(coeffs) % 2 == 1 and n >= 2
    K = (len(coeffs) - 1) // 2
    D = 2 * K + 1
    C = np.zeros((D, D_PHYS, D_PHYS, D))
    for cin in range(-K, K + 1):
        for w in range(D_PHYS):
            xb, yb = w >> 1, w & 1
            b = xb if direction == 1 else yb
            s = b + cin
            bin_ = s % 2
            cout = (s - bin_) // 2
            wp = (bin_ << 1 | yb) if direction == 1 else (xb << 1 | bin_)
            C[cout + K, w, wp, cin + K] = 1.0
    cores = [C.copy() for _ in range(n)]
    cores[0] = np.einsum("a,awvb->wvb", np.ones(D), C)[None]          # L on the most-significant end
    cores[-1] = np.einsum("awvb,b->awv", C, coeffs)[..., None]        # R on the least-significant end
    return cores


def fd_coefficients(order: int, dx: float):
    """Central first-derivative coefficients of even order 2, 4, 6, 8 for offsets -K..K (K = order / 2)."""
    table = {2: [0.5], 4: [2.0 / 3, -1.0 / 12], 6: [0.75, -0.15, 1.0 / 60], 8: [0.8, -0.2, 4.0 / 105, -1.0 / 280]}
    pos = table[order]
    return np.array([-c for c in pos[::-1]] + [0.0] + pos) / dx


def mpo_to_dense(W) -> np.ndarray:
    """Dense 4^n x 4^n matrix of an MPO in the (w_1..w_n) ordering (rows = output)."""
    M = W[0][0]  # (4,4,D)
    for Wk in W[1:]:
        M = np.einsum("opx,xqry->oqpry", M, Wk)
        o, q, p, r, y = M.shape
        M = M.reshape(o * q, p * r, y)
    return M[:, :, 0]


# --------------------------------------------------------------------------- O8
def rhs(u, Dx, Dy, Lap, Re, chi_max, eps=0.0, chi_work=None, skew=False, sketch_seed=None):
    """f_i = -(u_1 (.) D_1 u_i + u_2 (.) D_2 u_i) + (1/Re) Lap u_i, i = 1,2 (PAPER.md:49-53
    Eq. 2 without the pressure term; convective form, reading 4), with one rounding
    after every apply, product and sum (reading 7).

    skew=True: the paper's skew-symmetric convection (PAPER.md:432-435 Eq. B2),
    1/2 sum_j (u_j (.) D_j u_i + D_j (u_j (.) u_i)): in addition p_ij = round(u_j (.) u_i)
    (p_12 = p_21 computed once, as u_1 (.) u_2), d_ij = round(D_j p_ij), and
    f_i = round(-1/2 c_i1 - 1/2 c_i2 - 1/2 d_i1 - 1/2 d_i2 + (1/Re) Lap u_i) (one 5-term sum)."""
    Dj = (Dx, Dy)
    if skew:
        p11 = round_product(u[0], u[0], chi_max, eps, chi_work, sketch_seed=sketch_seed)
        p12 = round_product(u[0], u[1], chi_max, eps, chi_work, sketch_seed=sketch_seed)
        p22 = round_product(u[1], u[1], chi_max, eps, chi_work, sketch_seed=sketch_seed)
        pij = [[p11, p12], [p12, p22]]
    f = []
    for i in range(2):
        g = [round_mps(apply_mpo(Dj[j], u[i]), chi_max, eps) for j in range(2)]
        lap = round_mps(apply_mpo(Lap, u[i]), chi_max, eps)
        c = [round_product(u[j], g[j], chi_max, eps, chi_work, sketch_seed=sketch_seed) for j in range(2)]
        if skew:
            d = [round_mps(apply_mpo(Dj[j], pij[i][j]), chi_max, eps) for j in range(2)]
            terms = [(-0.5, c[0]), (-0.5, c[1]), (-0.5, d[0]), (-0.5, d[1]), (1.0 / Re, lap)]
        else:
            terms = [(-1.0, c[0]), (-1.0, c[1]), (1.0 / Re, lap)]
        f.append(round_mps(lincomb(terms), chi_max, eps))
    return f


# --------------------------------------------------------------------------- O9
def rk4_step(u, Dx, Dy, Lap, Re, dt, chi_max, eps=0.0, chi_work=None, skew=False, info=None, sketch_seed=None):
    """Classical RK4 (Eq. 11) on the MPS pair u = [u_1, u_2]; all
    roundings with the same (chi_max, eps); final combination as one 5-term sum
    and one rounding (reading 10).  ``info`` (a dict), if given, receives under "final" the two
    round_mps records (norm, singular values, discarded weight per bond) of the last rounding."""
    def stage(k, h):
        return [round_mps(lincomb([(1.0, u[i]), (h, k[i])]), chi_max, eps) for i in range(2)]

    k1 = rhs(u, Dx, Dy, Lap, Re, chi_max, eps, chi_work, skew, sketch_seed)
    k2 = rhs(stage(k1, dt / 2), Dx, Dy, Lap, Re, chi_max, eps, chi_work, skew, sketch_seed)
    k3 = rhs(stage(k2, dt / 2), Dx, Dy, Lap, Re, chi_max, eps, chi_work, skew, sketch_seed)
    k4 = rhs(stage(k3, dt), Dx, Dy, Lap, Re, chi_max, eps, chi_work, skew, sketch_seed)
    recs = [{}, {}] if info is not None else [None, None]
    out = [
        round_mps(
            lincomb([(1.0, u[i]), (dt / 6, k1[i]), (dt / 3, k2[i]), (dt / 3, k3[i]), (dt / 6, k4[i])]),
            chi_max, eps, recs[i])
        for i in range(2)
    ]
    if info is not None:
        info["final"] = recs
    return out


# ------------------------------------------------------------ harness utilities
def norm(cores) -> float:
    return math.sqrt(max(dot(cores, cores), 0.0))


def dot(A, B) -> float:
    """<A|B> by transfer matrices."""
    E = np.ones((1, 1))
    for a, b in zip(A, B):
        E = np.einsum("xy,xwa,ywb->ab", E, a, b, optimize=True)
    return float(E[0, 0])


def diff_norm(A, B) -> float:
    """||A - B||_F without cancellation: norm of the exact difference MPS obtained
    from a QR sweep (reading 19)."""
    D = _sweep_lr(lincomb([(1.0, A), (-1.0, B)]))
    return float(np.linalg.norm(D[-1]))


def schmidt_values(cores):
    """Singular values at every bond 1..n-1 (Eq. 16-17): SVD of the
    centre matrix while sweeping the orthogonality centre right-to-left."""
    C = _sweep_lr(cores)
    n = len(C)
    out = [None] * (n + 1)
    for k in range(n - 1, 0, -1):
        r0, d, r1 = C[k].shape
        U, s, Vt = np.linalg.svd(C[k].reshape(r0, d * r1), full_matrices=False)
        out[k] = s
        C[k] = Vt.reshape(len(s), d, r1)
        p0 = C[k - 1].shape[0]
        C[k - 1] = (C[k - 1].reshape(p0 * d, r0) @ (U * s)).reshape(p0, d, len(s))
    return out


def canonical_random(raw_cores):
    """BASELINE config 5: left-canonicalise raw random cores and scale the last
    core to unit norm."""
    C = _sweep_lr(raw_cores)
    C[-1] = C[-1] / np.linalg.norm(C[-1])
    return C


# ------------------------------------------------------- diagnostics
def fidelity(A, B) -> float:
    """F = <a|b>^2 / (||a||^2 ||b||^2)  (Eq. 12)."""
    na, nb = norm(A), norm(B)
    if na == 0.0 or nb == 0.0:
        return 0.0
    return dot(A, B) ** 2 / (na * na * nb * nb)


def tke_spectrum(u1, u2, mean1=None, mean2=None):
    """Turbulent-kinetic-energy spectrum (Eq. 13-15) of the velocity MPS pair (u1, u2):
    u_i' = u_i - mean_i (Eq. 14; mean_i = None: zero), Fourier coefficients u_i'^(k) = (1/N^2) sum_x u_i'(x) exp(-2 pi i k.x)
    on the N x N periodic grid, E(k1, k2) = 1/2 (|u_1'^|^2 + |u_2'^|^2) (Eq. 13), and E(kappa) = the sum of E(k1, k2) over the
    shell round(sqrt(k1^2 + k2^2)) = kappa (Eq. 15, the integral over the circle discretised to integer shells).
    Returns E[0 .. floor(N / sqrt(2) + 1/2)]; sum(E) = 1/2 mean(u_1'^2 + u_2'^2) (Parseval)."""
    f = []
    for u, m in ((u1, mean1), (u2, mean2)):
        F = to_dense(u)
        if m is not None:
            F = F - to_dense(m)
        f.append(F)
    N = f[0].shape[0]
    k = np.fft.fftfreq(N, d=1.0 / N)  # integer wave numbers -N/2 .. N/2-1
    K1, K2 = np.meshgrid(k, k, indexing="ij")
    shell = np.floor(np.sqrt(K1 * K1 + K2 * K2) + 0.5).astype(np.int64)
    E2 = 0.5 * sum(np.abs(np.fft.fft2(F) / (N * N)) ** 2 for F in f)
    nb = int(math.floor(math.sqrt(2.0) * (N // 2) + 0.5)) + 1
    return np.bincount(shell.reshape(-1), weights=E2.reshape(-1), minlength=nb)[:nb]


def chi_eps(cores, eps: float):
    """chi_l(eps) for every bipartition l = 1..n-1 and chi = max_l chi_l (Eq. 16-17): the
    number of Schmidt values needed so that the relative truncation error of that bipartition,
    sqrt(sum_{i > chi_l} sigma_i^2) / ||u||, is <= eps.  Returns ([1, chi_1, ..., chi_{n-1}, 1], chi)."""
    sv = schmidt_values(cores)
    n = len(cores)
    out = [1] * (n + 1)
    for k in range(1, n):
        s = np.asarray(sv[k], dtype=np.float64)
        tot = math.sqrt(float(np.sum(s[::-1] ** 2)))
        chi = len(s)
        for cand in range(len(s), 0, -1):
            tail = math.sqrt(float(np.sum(s[cand:][::-1] ** 2)))
            if tail <= eps * tot:
                chi = cand
            else:
                break
        out[k] = max(1, chi)
    return out, max(out)


# ------------------------------------------- variational stage (Sec. II.C, App. B)
def mpo_product(W1, W2):
    """MPO of the operator product W1 W2 (W1 acts after W2): cores [(m1,m2)][w][w''][(m1',m2')]."""
    out = []
    for A, B in zip(W1, W2):
        C = np.einsum("aopb,cpqd->acoqbd", A, B)
        a, c, o, q, b, d = C.shape
        out.append(C.reshape(a * c, o, q, b * d))
    return out


def variational_cost(v, a, Bm, D1, D2, h, mu):
    """Theta of PAPER.md:452 Eq. B6 with the nonlinear part given as the MPS pair B (Eq. B21):
    mu ||D1 v1 + D2 v2||^2 + sum_i ||(v_i - a_i)/h + B_i||^2, evaluated with exact MPS sums (no rounding)."""
    div = lincomb([(1.0, apply_mpo(D1, v[0])), (1.0, apply_mpo(D2, v[1]))])
    th = mu * float(np.linalg.norm(_sweep_lr(div)[-1])) ** 2
    for i in range(2):
        res = lincomb([(1.0 / h, v[i]), (-1.0 / h, a[i]), (1.0, Bm[i])])
        th += float(np.linalg.norm(_sweep_lr(res)[-1])) ** 2
    return th


def _canonicalize_right(cores):
    """Right-canonical form with the centre on site 1 (PAPER.md:498-518 Eq. B15-B19): QR sweeps only, bonds kept."""
    C = [c.copy() for c in cores]
    for k in range(len(C) - 1, 0, -1):
        r0, d, r1 = C[k].shape
        Q, R = np.linalg.qr(C[k].reshape(r0, d * r1).T)       # M^T = Q R  ->  M = R^T Q^T
        C[k] = Q.T.reshape(-1, d, r1)
        p0 = C[k - 1].shape[0]
        C[k - 1] = (C[k - 1].reshape(p0 * d, r0) @ R.T).reshape(p0, d, -1)
    return C


def variational_stage(v0, a, Bm, D1, D2, h, mu, max_sweeps=20, sweep_tol=1e-5, cg_maxit=100, cg_tol=1e-5, info=None):
    """One Euler-type stage of the paper's DMRG-like solver (Sec. II.C; App. B): minimise Theta (Eq. B6)
    over the trial MPS pair v (bonds of v0 kept) by one-site sweeps.  At the canonical centre d the stationarity condition
    Eq. B22 is the coupled linear system Eq. B23-B24,
        C_i - mu h^2 sum_j <basis_i| D_i D_j |basis_j> C_j = <basis_i| a_i - h B_i>,     i = 1, 2,
    (D^T = -D, so the operator is I + mu h^2 P^T (D^T D) P: symmetric positive definite), solved by
    conjugate gradients from the current centre tensors, at most cg_maxit iterations or until ||r|| <= cg_tol ||rhs||
    (100 iterations, 1e-5); the centre is then shifted by a QR factorisation and the environments are
    updated.  A sweep runs the centre from site 1 to site n and back; the iteration stops when the
    relative change of sum_i <v_i|v_i> between sweeps is below sweep_tol (1e-5 in the paper) or after max_sweeps.
    Reading: the nonlinear part B_i of Eq. B21 enters as an MPS (formed by the hot-path primitives: -rhs with
    the skew-symmetric convection), so its projection is a two-layer overlap instead of the paper's four-layer network."""
    n = len(v0[0])
    V = [_canonicalize_right(v0[0]), _canonicalize_right(v0[1])]
    Dm = (D1, D2)
    Wij = [[mpo_product(Dm[i], Dm[j]) for j in range(2)] for i in range(2)]
    g = [lincomb([(1.0, a[i]), (-h, Bm[i])]) for i in range(2)]
    # environments: LH[i][j][k] (r^i_k, m_k, r^j_k) of <v_i| D_i D_j |v_j> left of site k+1 / RH right of site k;
    # LG[i][k] (r^i_k, rg_k) of <v_i| g_i>
    one3, one2 = np.ones((1, 1, 1)), np.ones((1, 1))
    LH = [[[None] * (n + 1) for _ in range(2)] for _ in range(2)]
    RH = [[[None] * (n + 1) for _ in range(2)] for _ in range(2)]
    LG = [[None] * (n + 1) for _ in range(2)]
    RG = [[None] * (n + 1) for _ in range(2)]

    def upd_left(k):
        for i in range(2):
            for j in range(2):
                LH[i][j][k + 1] = np.einsum("amc,awb,mwxn,cxd->bnd", LH[i][j][k], V[i][k], Wij[i][j][k], V[j][k], optimize=True)
            LG[i][k + 1] = np.einsum("ac,awb,cwd->bd", LG[i][k], V[i][k], g[i][k], optimize=True)

    def upd_right(k):
        for i in range(2):
            for j in range(2):
                RH[i][j][k] = np.einsum("bnd,awb,mwxn,cxd->amc", RH[i][j][k + 1], V[i][k], Wij[i][j][k], V[j][k], optimize=True)
            RG[i][k] = np.einsum("bd,awb,cwd->ac", RG[i][k + 1], V[i][k], g[i][k], optimize=True)

    for i in range(2):
        for j in range(2):
            LH[i][j][0], RH[i][j][n] = one3, one3
        LG[i][0], RG[i][n] = one2, one2
    for k in range(n - 1, 0, -1):
        upd_right(k)

    cg_its = []

    def solve_site(d):
        def op(x):
            y = [x[0].copy(), x[1].copy()]
            for i in range(2):
                for j in range(2):
                    y[i] = y[i] - mu * h * h * np.einsum("amc,mwxn,bnd,cxd->awb", LH[i][j][d], Wij[i][j][d], RH[i][j][d + 1],
                                                         x[j], optimize=True)
            return y
        rhs_ = [np.einsum("ac,cwd,bd->awb", LG[i][d], g[i][d], RG[i][d + 1], optimize=True) for i in range(2)]
        dot2 = lambda p, q: float(np.sum(p[0] * q[0]) + np.sum(p[1] * q[1]))
        x = [V[0][d].copy(), V[1][d].copy()]
        Ax = op(x)
        r = [rhs_[i] - Ax[i] for i in range(2)]
        p = [r[0].copy(), r[1].copy()]
        rr = dot2(r, r)
        bnorm = math.sqrt(dot2(rhs_, rhs_))
        its = 0
        while its < cg_maxit and math.sqrt(rr) > cg_tol * bnorm:
            Ap = op(p)
            alpha = rr / dot2(p, Ap)
            for i in range(2):
                x[i] = x[i] + alpha * p[i]
                r[i] = r[i] - alpha * Ap[i]
            rr_new = dot2(r, r)
            beta = rr_new / rr
            for i in range(2):
                p[i] = r[i] + beta * p[i]
            rr = rr_new
            its += 1
        cg_its.append(its)
        V[0][d], V[1][d] = x[0], x[1]

    def shift_right(d):
        for i in range(2):
            r0, dd, r1 = V[i][d].shape
            Q, R = np.linalg.qr(V[i][d].reshape(r0 * dd, r1))
            V[i][d] = Q.reshape(r0, dd, -1)
            nr0, _, nr1 = V[i][d + 1].shape
            V[i][d + 1] = (R @ V[i][d + 1].reshape(nr0, dd * nr1)).reshape(-1, dd, nr1)

    def shift_left(d):
        for i in range(2):
            r0, dd, r1 = V[i][d].shape
            Q, R = np.linalg.qr(V[i][d].reshape(r0, dd * r1).T)
            V[i][d] = Q.T.reshape(-1, dd, r1)
            p0 = V[i][d - 1].shape[0]
            V[i][d - 1] = (V[i][d - 1].reshape(p0 * dd, r0) @ R.T).reshape(p0, dd, -1)

    norm2 = lambda: float(np.sum(V[0][0] ** 2) + np.sum(V[1][0] ** 2))
    prev = norm2()
    sweeps = 0
    for sweeps in range(1, max_sweeps + 1):
        for d in range(n - 1):
            solve_site(d)
            shift_right(d)
            upd_left(d)
        solve_site(n - 1)
        for d in range(n - 1, 0, -1):
            shift_left(d)
            upd_right(d)
            solve_site(d - 1)
        cur = norm2()
        change = abs(cur - prev) / max(cur, 1e-300)
        prev = cur
        if change < sweep_tol:
            break
    if info is not None:
        info["sweeps"] = sweeps
        info["cg_iterations"] = cg_its
    return V
