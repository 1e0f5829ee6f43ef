"""Dense 3V x 3V staggered Dirac matrix built from the definition, independently of oracle/.

Used only as a pin for the oracle (tests/test_oracle_pins.py).  Pure numpy + Python loops; no
code shared with oracle/ or with the CUDA path.  Definition (readings R1-R4):

  D[(x,a),(x+mu,b)] += 1/2 eta_mu(x) s+_mu(x)  U_mu(x)[a,b]
  D[(x,a),(x-mu,b)] -= 1/2 eta_mu(x) s-_mu(x)  conj(U_mu(x-mu)[b,a])

with eta_mu(x) = (-1)^(x_0+...+x_{mu-1}), periodic wrap, and s = -1 on the hop that crosses
the x3 boundary when antiperiodic_t.  '+=' (not '=') so that N_mu = 2, where x+mu == x-mu,
receives both contributions.
"""
import itertools

import numpy as np


def dense_dirac(dims, U, antiperiodic_t=True, theta=None):
    """theta[V][4] (optional): every link enters as exp(i theta_mu(x)) U_mu(x) (the backfield)."""
    if theta is not None:
        U = U * np.exp(1j * np.asarray(theta))[:, :, None, None]
    return _dense_dirac(dims, U, antiperiodic_t)


def _dense_dirac(dims, U, antiperiodic_t):
    n0, n1, n2, n3 = dims
    V = n0 * n1 * n2 * n3
    D = np.zeros((3 * V, 3 * V), dtype=np.complex128)
    N = (n0, n1, n2, n3)

    def lex(c):
        return c[0] + n0 * (c[1] + n1 * (c[2] + n2 * c[3]))

    for x3, x2, x1, x0 in itertools.product(range(n3), range(n2), range(n1), range(n0)):
        x = (x0, x1, x2, x3)
        i = lex(x)
        for mu in range(4):
            eta = (-1.0) ** sum(x[:mu])
            fwd = list(x)
            fwd[mu] = (x[mu] + 1) % N[mu]
            bwd = list(x)
            bwd[mu] = (x[mu] - 1) % N[mu]
            s_fwd = -1.0 if (antiperiodic_t and mu == 3 and x[3] == N[3] - 1) else 1.0
            s_bwd = -1.0 if (antiperiodic_t and mu == 3 and x[3] == 0) else 1.0
            jf, jb = lex(fwd), lex(bwd)
            D[3 * i:3 * i + 3, 3 * jf:3 * jf + 3] += 0.5 * eta * s_fwd * U[i, mu]
            D[3 * i:3 * i + 3, 3 * jb:3 * jb + 3] -= 0.5 * eta * s_bwd * U[jb, mu].conj().T
    return D


def parity_mask(dims):
    """mask[lex] = (x0+x1+x2+x3) % 2."""
    n0, n1, n2, n3 = dims
    x0, x1, x2, x3 = np.meshgrid(np.arange(n0), np.arange(n1), np.arange(n2), np.arange(n3), indexing="ij")
    par = (x0 + x1 + x2 + x3) % 2
    # lex = x0 + n0*(x1 + ...): x0 fastest -> transpose to (x3,x2,x1,x0) and ravel C-order
    return par.transpose(3, 2, 1, 0).reshape(-1)


def dense_normal_operator(dims, U, mass, antiperiodic_t=True, theta=None):
    """A = m^2 - D_eo D_oe on even sites, as a (3 Vh) x (3 Vh) matrix in idxh order."""
    D = dense_dirac(dims, U, antiperiodic_t, theta)
    par = np.repeat(parity_mask(dims), 3)
    even = np.nonzero(par == 0)[0]
    odd = np.nonzero(par == 1)[0]
    D_oe = D[np.ix_(odd, even)]   # output odd, input even
    D_eo = D[np.ix_(even, odd)]   # output even, input odd
    return mass * mass * np.eye(even.size) - D_eo @ D_oe, D_eo, D_oe
