"""CPU oracle of the paper's OWN recursion: the tensor-based free-energy model with a codon tensor train.

Test infrastructure, NOT the product: only tests/ may import this module; it shares no code with the CUDA path
(paper_2604_19718_b200/csrc/cdz_tm.cu) and never imports it.  Plain numpy fp64, one small matrix product per term, in the
order of the paper's Algorithm S4.1; nothing is blocked, fused, scaled or reordered.

What is computed:
  eq 3.5 (line 171)   Q_{i,j} = sum_{k in [i:j)} Q_{i,k} Q_{j,k}^T  (i < j),   Q_{i,j} = chi_{j,i}(Q_{j+1,i-1})  (i >= j)
  eq 3.6 (line 178)   chi_{i,j+1}(X) = I (i = j+1) | V_i^T (i = j) | sum_rho B_{i,j}^{rho,T} Tr_S[B_{j,i}^rho X]  (otherwise)
  eq 3.7 (line 184)   Z = Tr_S[ Q_{0,n} ]   (the printed sum over k of Tr_S[Q_{0,k} chi^T_{k,n}(..)] is Q_{0,n} by eq 3.5)
  eq 3.8 (lines 203-209)  chi-hat: the same with every V / B dressed by the tensor-train cores T_i of the summed nucleotides; a block
                      Q_{i,j} becomes a (gamma Sigma_i) x (gamma Sigma_j) matrix, flattened (sigma, zeta) -> sigma * gamma + zeta
  Alg S4.1 (lines 586-601) loop order.
Indices are boundary points 0..n; Q_{i,j} with i < j ("upper") is the backbone product over the half-open interval [i:j); Q_{j,k}
with j > k ("lower") is the transposed closed element over exactly [k:j): the unpaired base k when j = k+1, else the base pair
k.(j-1) around the interval [k+1:j-1).  Tr_S[X] = Tr[S X] (line 178).

Readings: (i) a pair k.l needs l - k - 1 >= min_hairpin (line 483); (ii) open chain: left bond Sigma_0 = 1,
the last bond is summed out (lines 561-567) -- Z = sum_{sigma_n} Tr_S of that block of Q_{0,n}; (iii) B[x][y] is the tensor of the 5'
side of a pair whose 5' base is x and 3' base y ("B_{i,j}"), B[y][x] the tensor of its 3' side ("B_{j,i}"); a zero tensor means x.y
cannot pair; (iv) the parameters are synthetic and non-negative -- the cyclic symmetry that ref [15] builds into S is not needed by
the recursion and not imposed.

`tm_brute_force` is the definition the recursion must reproduce: explicit enumeration of every coding sequence (operator path) and
every unpseudoknotted structure, each state contracted as its own tensor diagram (eq S2.1 / S2.2, lines 439-446: every loop is the
Tr_S of the product of the matrices along its backbone, the two tensors of a pair share one conformation index rho).
"""
from __future__ import annotations

import math

import numpy as np


def cores(sigma, ops):
    """Dense tensor-train cores T[p][x] (Sigma_p x Sigma_{p+1}) = sum of the operator weights (eq S3.7)."""
    T = []
    for p, lst in enumerate(ops):
        t = np.zeros((4, sigma[p], sigma[p + 1]))
        for (a, b, c, x) in lst:
            t[b, a, c] += x
        T.append(t)
    return T


def chi_hat(tm, sigma, T, i, j, Q):
    """The lower block Q_{j,i} = chi-hat_{i,j} of eq 3.8 for boundary points i <= j, as a (gamma Sigma_j) x (gamma Sigma_i) matrix."""
    g = tm.gamma
    if i == j:
        return np.eye(g * sigma[i])
    if j == i + 1:
        # unpaired base i: sum_x T_i[x] (x) V[x], transposed (eq 3.6 second case)
        C = np.zeros((g * sigma[i], g * sigma[j]))
        for x in range(4):
            C += np.kron(T[i][x], tm.V[x])
        return C.T
    C = np.zeros((g * sigma[i], g * sigma[j]))
    k, l = i, j - 1  # the pair k.l
    if l - k - 1 >= tm.min_hairpin:
        X = Q[k + 1][l]  # backbone product over the enclosed interval [k+1 : l)
        for x in range(4):
            for y in range(4):
                for sa in range(sigma[k]):
                    for sb in range(sigma[k + 1]):
                        tk = T[k][x][sa, sb]
                        if tk == 0.0:
                            continue
                        for sc in range(sigma[l]):
                            Xb = X[sb * g:(sb + 1) * g, sc * g:(sc + 1) * g]
                            for sd in range(sigma[l + 1]):
                                tl = T[l][y][sc, sd]
                                if tl == 0.0:
                                    continue
                                for rho in range(tm.xi):
                                    tr = np.trace(tm.S @ tm.B[y][x][rho] @ Xb)  # Tr_S[B_{j,i}^rho X]
                                    C[sa * g:(sa + 1) * g, sd * g:(sd + 1) * g] += tk * tl * tr * tm.B[x][y][rho]
    return C.T


def tm_inside(tm, sigma, ops, return_Q: bool = False):
    """log Z by Algorithm S4.1 (AbstractFreeEnergy with chi-hat); optionally the whole block matrix Q."""
    n, g = len(ops), tm.gamma
    T = cores(sigma, ops)
    Q = [[None] * (n + 1) for _ in range(n + 1)]
    for j in range(n + 1):
        for i in range(j + 1):
            Q[j][i] = chi_hat(tm, sigma, T, i, j, Q)
        for i in range(j):
            acc = np.zeros((g * sigma[i], g * sigma[j]))
            for k in range(i, j):
                acc += Q[i][k] @ Q[j][k].T
            Q[i][j] = acc
    Z = 0.0
    for s in range(sigma[n]):
        Z += np.trace(tm.S @ Q[0][n][0:g, s * g:(s + 1) * g])
    logZ = math.log(Z)
    return (logZ, Q) if return_Q else logZ


def _structures(n, can_pair, mh):
    """Every unpseudoknotted pair table of n bases (partner or -1) whose pairs satisfy can_pair(k, l) and l - k - 1 >= mh."""
    def rec(a, b):
        # all structures of the interval [a:b) as lists of pairs
        if b - a <= 0:
            yield []
            return
        for rest in rec(a + 1, b):  # base a unpaired
            yield rest
        for l in range(a + mh + 1, b):  # base a paired with l
            if not can_pair(a, l):
                continue
            for inner in rec(a + 1, l):
                for rest in rec(l + 1, b):
                    yield [(a, l)] + inner + rest
    for pairs in rec(0, n):
        pt = [-1] * n
        for (k, l) in pairs:
            pt[k], pt[l] = l, k
        yield pt


def state_weight(tm, seq, pt):
    """Tr_S of the exterior backbone product of one (sequence, structure) state: the tensor diagram of eq S2.1 contracted loop by loop."""
    g = tm.gamma

    def seg(a, b):
        M = np.eye(g)
        p = a
        while p < b:
            if pt[p] < 0:
                M = M @ tm.V[seq[p]]
                p += 1
            else:
                l = pt[p]
                inner = seg(p + 1, l)
                E = np.zeros((g, g))
                for rho in range(tm.xi):
                    E += tm.B[seq[p]][seq[l]][rho] * np.trace(tm.S @ tm.B[seq[l]][seq[p]][rho] @ inner)
                M = M @ E
                p = l + 1
        return M

    return float(np.trace(tm.S @ seg(0, len(seq))))


def tm_brute_force(tm, sigma, ops):
    """(log Z, number of states) by explicit enumeration of operator paths x structures."""
    n = len(ops)
    paths = []  # (sequence, weight)

    def walk(p, bond, seq, w):
        if p == n:
            paths.append((list(seq), w))
            return
        for (a, b, c, x) in ops[p]:
            if a == bond:
                seq.append(b)
                walk(p + 1, c, seq, w * x)
                seq.pop()

    walk(0, 0, [], 1.0)
    Z, ns = 0.0, 0
    for seq, w in paths:
        def can_pair(k, l, seq=seq):
            return bool(np.any(tm.B[seq[k]][seq[l]] != 0.0))
        for pt in _structures(n, can_pair, tm.min_hairpin):
            Z += w * state_weight(tm, seq, pt)
            ns += 1
    return math.log(Z), ns


# decision kinds of the tensor-model traceback (distinct from the kinds 0..8 of the nearest-neighbour traceback)
TMK_TOP, TMK_UPPER, TMK_UNPAIRED, TMK_PAIR = 16, 17, 18, 19


def _pick(alts, total, u):
    """First alternative whose running sum exceeds u * total; zero-weight alternatives are skipped; if rounding leaves the threshold above
    the last running sum the last positive alternative is taken (the rule of DESIGN.md section 5)."""
    thr, run, last = u * total, 0.0, None
    for key, w in alts:
        if not (w > 0.0):
            continue
        run += w
        last = key
        if run > thr:
            return key
    return last


def tm_sample(tm, sigma, ops, Q, J, seed, uniform):
    """J exact samples (sequence, structure) ~ W(phi) Z(phi, s) / Z by stochastic traceback of the block matrix Q (section 4a
    lines 215-217; the alternatives are those of Alg S4.4, taken per sample -- the simultaneous bookkeeping of Alg S4.4 changes
    the cost, not the distribution).  One uniform per decision, uniform(seed, sample, kind, i, j); `total` is the stored block entry being
    decomposed.  Recursion elements and their alternatives, in this order:
      TOP                    (s, d, e) ascending:  S[d][e] Q_{0,n}[(0,e)][(s,d)]                                -> UPPER(0, n, (0,e), (s,d))
      UPPER(i,j,a,b), i < j  k in [i:j) ascending, c ascending:  Q_{i,k}[a][c] Q_{j,k}[b][c]                    -> UPPER(i,k,a,c) if k > i, LOWER(j,k,b,c)
      LOWER(j,k,b,c), j = k+1   x ascending:  T_k[x][sigma(c)][sigma(b)] V[x][zeta(c)][zeta(b)]                  -> base k = x
      LOWER(j,k,b,c), j > k+1   (x, y, s1, s2, rho, cc, dd) ascending, l = j-1:
                             T_k[x][sigma(c)][s1] T_l[y][s2][sigma(b)] B[x][y][rho][zeta(c)][zeta(b)] (S B[y][x][rho])[dd][cc] Q_{k+1,l}[(s1,cc)][(s2,dd)]
                                                                                                                -> pair k.l, UPPER(k+1, l, (s1,cc), (s2,dd))
    Nucleotides are chosen through the dense cores (operators with the same (a, b, c) are one alternative).  Returns (seq [J][n] uint8,
    pair [J][n] int32 with -1 = unpaired)."""
    n, g = len(ops), tm.gamma
    T = cores(sigma, ops)
    SB = np.zeros_like(tm.B)
    for y in range(4):
        for x in range(4):
            for rho in range(tm.xi):
                SB[y][x][rho] = tm.S @ tm.B[y][x][rho]
    seqs = np.full((J, n), 255, dtype=np.uint8)
    pairs = np.full((J, n), -1, dtype=np.int32)
    for smp in range(J):
        alts = []
        for s in range(sigma[n]):
            for d in range(g):
                for e in range(g):
                    alts.append(((e, s * g + d), tm.S[d, e] * Q[0][n][e, s * g + d]))
        a, b = _pick(alts, sum(w for _, w in alts if w > 0.0), uniform(seed, smp, TMK_TOP, 0, 0))
        stack = [("U", 0, n, a, b)]
        while stack:
            kind, i, j, a, b = stack.pop()
            if kind == "U":
                if i == j:
                    continue
                alts = []
                for k in range(i, j):
                    for c in range(g * sigma[k]):
                        alts.append(((k, c), Q[i][k][a, c] * Q[j][k][b, c]))
                k, c = _pick(alts, Q[i][j][a, b], uniform(seed, smp, TMK_UPPER, i, j))
                if k > i:
                    stack.append(("U", i, k, a, c))
                stack.append(("L", j, k, b, c))
            else:
                j, k, b, c = i, j, a, b  # the item is ("L", j, k, b, c)
                if j == k + 1:
                    alts = [(x, T[k][x][c // g, b // g] * tm.V[x][c % g, b % g]) for x in range(4)]
                    x = _pick(alts, Q[j][k][b, c], uniform(seed, smp, TMK_UNPAIRED, k, j))
                    seqs[smp, k] = x
                else:
                    l = j - 1
                    alts = []
                    for x in range(4):
                        for y in range(4):
                            for s1 in range(sigma[k + 1]):
                                tk = T[k][x][c // g, s1]
                                for s2 in range(sigma[l]):
                                    tl = T[l][y][s2, b // g]
                                    for rho in range(tm.xi):
                                        bo = tm.B[x][y][rho][c % g, b % g]
                                        for cc in range(g):
                                            for dd in range(g):
                                                alts.append(((x, y, s1, s2, cc, dd),
                                                             tk * tl * bo * SB[y][x][rho][dd, cc] * Q[k + 1][l][s1 * g + cc, s2 * g + dd]))
                    x, y, s1, s2, cc, dd = _pick(alts, Q[j][k][b, c], uniform(seed, smp, TMK_PAIR, k, j))
                    seqs[smp, k], seqs[smp, l] = x, y
                    pairs[smp, k], pairs[smp, l] = l, k
                    stack.append(("U", k + 1, l, s1 * g + cc, s2 * g + dd))
    return seqs, pairs


def tm_state_distribution(tm, sigma, ops):
    """Exact distribution over (sequence, structure) by enumeration: {(seq tuple, pair tuple): probability}."""
    n = len(ops)
    paths = []

    def walk(p, bond, seq, w):
        if p == n:
            paths.append((tuple(seq), w))
            return
        for (a, b, c, x) in ops[p]:
            if a == bond:
                seq.append(b)
                walk(p + 1, c, seq, w * x)
                seq.pop()

    walk(0, 0, [], 1.0)
    dist, Z = {}, 0.0
    for seq, w in paths:
        def can_pair(k, l, seq=seq):
            return bool(np.any(tm.B[seq[k]][seq[l]] != 0.0))
        for pt in _structures(n, can_pair, tm.min_hairpin):
            v = w * state_weight(tm, list(seq), pt)
            key = (seq, tuple(pt))
            dist[key] = dist.get(key, 0.0) + v
            Z += v
    return {k: v / Z for k, v in dist.items()}
