"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

The N-shaped partition method written out stage by stage in the paper's order and
notation (RD, JD, RU, JU, RS, SS), in complex128, as slow pure-Python loops for
small systems.  It exists so that a reader can check the *method* against the
paper by eye and so that tests can pin the structural claims of the paper
(stacked-N sparsity, reduced system size, exactness against Thomas / dense LU).
It shares no code with the CUDA path and is not used for ψ parity of the CUDA
path (that is `cn_oracle.step`, the plain definition).

Sources: PAPER.md:90-124 (§4.1.1-4.1.5), PAPER.md:106 (Fig. 1 caption),
PAPER.md:298-337 (Appendix I), PAPER.md:177-187 (stage order (RD+JD)+(RU+JU)).

Table 1 itself is lost in the extraction (only its caption survives,
PAPER.md:132); the body below is the reconstruction of SURVEY.md §8(c) /
DESIGN.md reading R1.  Appendix I prints the downward multiplier as
r_i = -T_{i,i-1}/T_{i,i}; that is a typo (reading R2): elimination
of T_{i,i-1} with row i-1 needs r_i = -T_{i,i-1}/T_{i-1,i-1}, the mirror image of
the upward one r_i = -T_{i,i+1}/T_{i+1,i+1} which is printed correctly
(PAPER.md:321).  tests/test_oracle_pins.py::test_table1_typo shows the printed form
does not solve the system and the corrected one does.

Indices in this file are the paper's 1-based row numbers; arrays are padded with
an unused element 0 so that a[i] is the paper's a_i.
"""
from __future__ import annotations

import numpy as np


def joints_paper(n_tot: int, n_bl: int):
    """J_0 = 1 < J_1 < ... < J_{n_bl} = n_tot; blocks may differ in size."""
    J = [1 + (w * (n_tot - 1)) // n_bl for w in range(n_bl + 1)]
    assert J[0] == 1 and J[-1] == n_tot and all(J[w + 1] > J[w] for w in range(n_bl))
    return J


def joints_uniform(n_tot: int, n_bl: int):
    """The CUDA path's layout (reading R8): the system is padded with one identity row 0
    (psi_0 = 0, the reflecting boundary of PAPER.md:84), joints are rows m, 2m, ..., n_tot and the
    virtual row 0.  Returned for the PADDED system of n_tot + 1 rows: J = [1, m+1, 2m+1, ...]."""
    assert n_tot % n_bl == 0
    m = n_tot // n_bl
    return [1] + [w * m + 1 for w in range(1, n_bl + 1)]


def _pad(v):
    v = np.asarray(v)
    if v.dtype == object:                      # instrumented scalars (operation counting in the tests)
        return np.concatenate([np.array([v[0] * 0], dtype=object), v])
    return np.concatenate([[0], np.asarray(v, dtype=np.complex128)])


def _zeros(shape, like):
    if like.dtype == object:
        z = np.empty(shape, dtype=object)
        z[...] = like[0] * 0
        return z
    return np.zeros(shape, np.complex128)


def solve(b, a, c, d, J, multiplier: str = "corrected"):
    """Run RD+JD, RU+JU, RS, SS on the tridiagonal system (b, a, c, d) with joint lines J.

    Returns (psi, state) with state = dict of the arrays after JU (1-based, padded) and the
    reduced system, so tests can look at the intermediate structure."""
    n = len(a)
    b, a, c, d = _pad(b), _pad(a), _pad(c), _pad(d)
    b[1] = 0.0
    c[n] = 0.0
    nbl = len(J) - 1
    # two extra elements per joint line instead of atomics: (a, d) contributions
    # from the block above (JD) and from the block below (JU), summed afterwards.
    extra_a = _zeros((nbl + 1, 2), a)
    extra_d = _zeros((nbl + 1, 2), a)
    for w in range(nbl):                       # "for all parallel processes w = 0..n_bl-1"
        Jw, Jn = J[w], J[w + 1]
        if Jn - Jw < 2:
            continue                           # no interior row: nothing to do
        # RD: downward elimination, fill-in goes to column J_w and is stored in b (Eq. 10-11)
        for i in range(Jw + 2, Jn):
            if multiplier == "corrected":
                r = -b[i] / a[i - 1]
            else:                              # as printed in PAPER.md:311
                r = -b[i] / a[i]
            a[i] = a[i] + r * c[i - 1]
            b[i] = r * b[i - 1]
            d[i] = d[i] + r * d[i - 1]
        # JD: contribution to the lower joint line
        i = Jn
        r = -b[i] / a[i - 1]
        extra_a[w + 1, 0] = r * c[i - 1]
        b[i] = r * b[i - 1]
        extra_d[w + 1, 0] = r * d[i - 1]
        # RU: upward elimination with the diagonal as modified by RD; fill-in to column J_{w+1}, stored in c
        for i in range(Jn - 2, Jw, -1):
            r = -c[i] / a[i + 1]
            b[i] = b[i] + r * b[i + 1]
            c[i] = r * c[i + 1]
            d[i] = d[i] + r * d[i + 1]
        # JU: contribution to the upper joint line
        i = Jw
        r = -c[i] / a[i + 1]
        extra_a[w, 1] = r * b[i + 1]
        c[i] = r * c[i + 1]
        extra_d[w, 1] = r * d[i + 1]
    for w in range(nbl + 1):                   # the deferred "atomic" additions
        a[J[w]] += extra_a[w, 0] + extra_a[w, 1]
        d[J[w]] += extra_d[w, 0] + extra_d[w, 1]
    # RS: the joint lines form a tridiagonal system of size n_bl + 1
    rb = np.array([b[j] for j in J]); ra = np.array([a[j] for j in J])
    rc = np.array([c[j] for j in J]); rd = np.array([d[j] for j in J])
    ra_f, rd_f = ra.copy(), rd.copy()
    for k in range(1, nbl + 1):                # e_d / f_d on the joint lines
        r = -rb[k] / ra_f[k - 1]
        ra_f[k] = ra_f[k] + r * rc[k - 1]
        rd_f[k] = rd_f[k] + r * rd_f[k - 1]
    sup = _zeros(nbl + 1, a)
    sup[nbl] = rd_f[nbl] / ra_f[nbl]
    for k in range(nbl - 1, -1, -1):
        sup[k] = (rd_f[k] - rc[k] * sup[k + 1]) / ra_f[k]
    # SS: psi_i = (d_i - b_i psi_{J_w} - c_i psi_{J_{w+1}}) / a_i, independent per row
    # The division is done once per row as 1/a_i and applied as a multiplication ("the precomputed values of
    # 1/a_i"); this is what gives the 3 divisions / 9 multiplications / 6 additions per row of
    # PAPER.md:215.
    psi = _zeros(n + 1, a)
    for w in range(nbl + 1):
        psi[J[w]] = sup[w]
    for w in range(nbl):
        for i in range(J[w] + 1, J[w + 1]):
            inv_a = 1.0 / a[i]
            psi[i] = (d[i] - b[i] * sup[w] - c[i] * sup[w + 1]) * inv_a
    state = dict(b=b, a=a, c=c, d=d, J=list(J), reduced=(rb, ra, rc, rd), support=sup)
    return psi[1:], state


def dense_after_joining(T, J):
    """Apply the RD/JD/RU/JU row operations to a DENSE copy of T (no knowledge of the band), so that
    the stacked-N sparsity of PAPER.md:110 / Fig. 1d can be asserted rather than assumed."""
    n = T.shape[0]
    M = np.zeros((n + 1, n + 1), np.complex128)
    M[1:, 1:] = T
    nbl = len(J) - 1
    orig = M.copy()
    add = []                                   # deferred joint-row additions (row, vector)
    for w in range(nbl):
        Jw, Jn = J[w], J[w + 1]
        if Jn - Jw < 2:
            continue
        for i in range(Jw + 2, Jn):
            r = -M[i, i - 1] / M[i - 1, i - 1]
            M[i, :] = M[i, :] + r * M[i - 1, :]
        r = -orig[Jn, Jn - 1] / M[Jn - 1, Jn - 1]
        add.append((Jn, r * M[Jn - 1, :].copy()))
        for i in range(Jn - 2, Jw, -1):
            r = -M[i, i + 1] / M[i + 1, i + 1]
            M[i, :] = M[i, :] + r * M[i + 1, :]
        r = -orig[Jw, Jw + 1] / M[Jw + 1, Jw + 1]
        add.append((Jw, r * M[Jw + 1, :].copy()))
    for row, vec in add:
        M[row, :] += vec
    return M[1:, 1:]
