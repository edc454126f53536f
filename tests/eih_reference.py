"""Independent literature reference used ONLY to pin the oracle: the full N-body first-order
post-Newtonian (Einstein-Infeld-Hoffmann) acceleration and conserved energy for point masses,
in harmonic coordinates, evaluated in mpmath multi-precision arithmetic for tiny N.

This is NOT the paper's limited method (it is the O(N^3) parent theory the paper truncates,
PAPER.md:37, refs [13, 14]); it shares nothing with oracle/ or the CUDA path.

  a_A = sum_{B!=A} G m_B n_BA / r_AB^2
      + (1/c^2) sum_{B!=A} (G m_B n_BA / r_AB^2) [ v_A^2 + 2 v_B^2 - 4 v_A.v_B - (3/2)(n_AB.v_B)^2
              - 4 sum_{C!=A} G m_C / r_AC - sum_{C!=B} G m_C / r_BC + (1/2) (x_B - x_A).a_B ]
      + (1/c^2) sum_{B!=A} (G m_B / r_AB^2) [ n_AB.(4 v_A - 3 v_B) ] (v_A - v_B)
      + (7 / (2 c^2)) sum_{B!=A} G m_B a_B / r_AB
  (n_AB = (x_A - x_B)/r_AB, n_BA = -n_AB, a_B = Newtonian acceleration of B inside 1PN terms)

  E = sum 1/2 m v^2 - 1/2 sum_{a!=b} G m_a m_b / r
    + (1/c^2) { 3/8 sum m v^4 + 1/4 sum_{a!=b} (G m_a m_b / r)[6 v_a^2 - 7 v_a.v_b - (n.v_a)(n.v_b)]
                + 1/2 sum_a sum_{b!=a} sum_{c!=a} G^2 m_a m_b m_c / (r_ab r_ac) }
"""
from mpmath import mp, mpf, sqrt

mp.dps = 50


def _v(a):
    return [mpf(t) for t in a]


def _dot(a, b):
    return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]


def _sub(a, b):
    return [a[0] - b[0], a[1] - b[1], a[2] - b[2]]


def newton_acc(m, x, G):
    n = len(m)
    out = []
    for a in range(n):
        acc = [mpf(0)] * 3
        for b in range(n):
            if b == a:
                continue
            d = _sub(x[b], x[a])
            r = sqrt(_dot(d, d))
            acc = [acc[k] + G * m[b] * d[k] / r**3 for k in range(3)]
        out.append(acc)
    return out


def eih_acc(m, x, v, G, c):
    """Full EIH accelerations; m, x, v are lists (mpf-convertible); returns list of [ax, ay, az] mpf."""
    m = _v(m)
    x = [_v(p) for p in x]
    v = [_v(p) for p in v]
    G, c2 = mpf(G), mpf(c) ** 2
    n = len(m)
    aN = newton_acc(m, x, G)

    def r_(a, b):
        d = _sub(x[a], x[b])
        return sqrt(_dot(d, d))

    out = []
    for A in range(n):
        acc = list(aN[A])
        for B in range(n):
            if B == A:
                continue
            r = r_(A, B)
            nAB = [t / r for t in _sub(x[A], x[B])]
            nBA = [-t for t in nAB]
            sA = sum(G * m[C] / r_(A, C) for C in range(n) if C != A)
            sB = sum(G * m[C] / r_(B, C) for C in range(n) if C != B)
            br = (_dot(v[A], v[A]) + 2 * _dot(v[B], v[B]) - 4 * _dot(v[A], v[B]) - mpf(3) / 2 * _dot(nAB, v[B]) ** 2
                  - 4 * sA - sB + mpf(1) / 2 * _dot(_sub(x[B], x[A]), aN[B]))
            w = [4 * v[A][k] - 3 * v[B][k] for k in range(3)]
            vAB = _sub(v[A], v[B])
            for k in range(3):
                acc[k] += (G * m[B] * nBA[k] / r**2) * br / c2
                acc[k] += (G * m[B] / r**2) * _dot(nAB, w) * vAB[k] / c2
                acc[k] += mpf(7) / 2 * G * m[B] * aN[B][k] / r / c2
        out.append(acc)
    return out


def eih_energy(m, x, v, G, c):
    m = _v(m)
    x = [_v(p) for p in x]
    v = [_v(p) for p in v]
    G, c2 = mpf(G), mpf(c) ** 2
    n = len(m)

    def r_(a, b):
        d = _sub(x[a], x[b])
        return sqrt(_dot(d, d))

    E0 = sum(m[a] * _dot(v[a], v[a]) / 2 for a in range(n))
    E1 = sum(mpf(3) / 8 * m[a] * _dot(v[a], v[a]) ** 2 for a in range(n))
    for a in range(n):
        for b in range(n):
            if b == a:
                continue
            r = r_(a, b)
            nab = [t / r for t in _sub(x[a], x[b])]
            E0 -= G * m[a] * m[b] / r / 2
            E1 += (G * m[a] * m[b] / r) / 4 * (6 * _dot(v[a], v[a]) - 7 * _dot(v[a], v[b]) - _dot(nab, v[a]) * _dot(nab, v[b]))
            for cc in range(n):
                if cc == a:
                    continue
                E1 += G * G * m[a] * m[b] * m[cc] / (r * r_(a, cc)) / 2
    return E0 + E1 / c2


def eih_momentum(m, x, v, G, c):
    """1PN total momentum of the EIH theory: sum m v (1 + v^2/2c^2) - (1/2c^2) sum_{a!=b} (G m_a m_b / r)[v_a + (v_a.n) n]."""
    m = _v(m)
    x = [_v(p) for p in x]
    v = [_v(p) for p in v]
    G, c2 = mpf(G), mpf(c) ** 2
    n = len(m)
    P = [mpf(0)] * 3
    for a in range(n):
        v2 = _dot(v[a], v[a])
        P = [P[k] + m[a] * v[a][k] * (1 + v2 / (2 * c2)) for k in range(3)]
        for b in range(n):
            if b == a:
                continue
            d = _sub(x[a], x[b])
            r = sqrt(_dot(d, d))
            nab = [t / r for t in d]
            P = [P[k] - G * m[a] * m[b] / r * (v[a][k] + _dot(v[a], nab) * nab[k]) / (2 * c2) for k in range(3)]
    return P
