"""Independent 4-dimensional tensor algebra used to pin the oracle's 3+1 formulas.

Nothing here restates the oracle's 3+1 expressions: everything is built from the covariant
definitions the paper prints (eqs. 1-2): the 4-metric assembled from (alpha, beta^i,
gamma_ij), u^mu, b^mu, T^{mu nu} = (rho h + b^2) u u + (p + b^2/2) g - b b, the dual Faraday tensor
*F^{mu nu} = b^mu u^nu - b^nu u^mu, and Christoffel symbols from metric derivatives.
"""
import numpy as np

SYM = [(0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2)]


def gamma3(met10):
    met10 = np.asarray(met10)
    g = np.zeros((3, 3), dtype=met10.dtype)
    for c, (i, j) in enumerate(SYM):
        g[i, j] = g[j, i] = met10[4 + c]
    return g


def metric4(met10):
    al, be, g = met10[0], np.asarray(met10[1:4]), gamma3(met10)
    bl = g @ be
    G = np.zeros((4, 4), dtype=g.dtype)
    G[0, 0] = -al * al + be @ bl
    G[0, 1:] = G[1:, 0] = bl
    G[1:, 1:] = g
    return G


def fluid4(prim9, met10, Gam):
    """u^mu, b^mu, T^{mu nu}, *F^{mu nu}, from the covariant definitions."""
    rho, ut, p, B = prim9[0], np.asarray(prim9[1:4]), prim9[4], np.asarray(prim9[5:8])
    al, be, g = met10[0], np.asarray(met10[1:4]), gamma3(met10)
    G = metric4(met10)
    Gi = np.linalg.inv(G)
    W = np.sqrt(1 + ut @ g @ ut)
    v = ut / W
    n_up = np.array([1 / al, *(-be / al)])          # unit normal n^mu
    u = W * (n_up + np.array([0, *v]))               # u^mu = W (n^mu + v^mu)
    Bfour = np.array([0, *B])                        # B^mu, spatial
    ul = G @ u
    # b^mu = P^mu_nu B^nu / W with P = delta + u u_  (projection of B orthogonal to u)
    b = (Bfour + u * (ul @ Bfour)) / W
    b2 = b @ G @ b
    h = 1 + Gam / (Gam - 1) * p / rho
    T = (rho * h + b2) * np.outer(u, u) + (p + b2 / 2) * Gi - np.outer(b, b)
    F = np.outer(b, u) - np.outer(u, b)
    return dict(u=u, b=b, b2=b2, T=T, Fdual=F, G=G, Gi=Gi, W=W, v=v, h=h)


def christoffel(G, dG):
    """Gamma^l_{mk} from g_{mu nu} and dG[k, mu, nu] = d_k g_{mu nu}."""
    Gi = np.linalg.inv(G)
    Gam = np.zeros((4, 4, 4))
    for l in range(4):
        for m in range(4):
            for k in range(4):
                s = 0.0
                for r in range(4):
                    s += Gi[l, r] * (dG[k, r, m] + dG[m, r, k] - dG[r, m, k])
                Gam[l, m, k] = 0.5 * s
    return Gam
