"""Independent reference formulas used ONLY by the tests to pin the oracle: fluxes and conserved
variables written straight from the covariant definitions (Eqs. 1-3, 5, 7; lines 51-101)
with the full 4-metric — none of the 3+1 forms of Eq. 8 that the oracle restates."""
import numpy as np

SYM = ((0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2))


def sym6_to_mat(g6):
    m = np.zeros((3, 3))
    for q, (i, j) in enumerate(SYM):
        m[i, j] = m[j, i] = g6[q]
    return m


def random_spd(rng, strength=0.3):
    a = np.eye(3) + strength * rng.uniform(-1, 1, (3, 3))
    m = a @ a.T
    return np.array([m[i, j] for (i, j) in SYM])


def tensor_state(alpha, beta_u, g6, rho, v_u, P, B_u, Gamma, h=None):
    """Conserved (D,S_i,tau,B^i) and flux matrices F[j] (j = direction) of
    (D,S_x,S_y,S_z,tau,B^x,B^y,B^z), all multiplied by sqrt(gamma), from T^{mu nu}, *F^{mu nu}."""
    gam = sym6_to_mat(g6)
    beta_u = np.asarray(beta_u, float); v_u = np.asarray(v_u, float); B_u = np.asarray(B_u, float)
    beta_l = gam @ beta_u
    g4 = np.zeros((4, 4))
    g4[0, 0] = -alpha ** 2 + beta_l @ beta_u
    g4[0, 1:] = g4[1:, 0] = beta_l
    g4[1:, 1:] = gam
    g4i = np.linalg.inv(g4)
    sg = np.sqrt(np.linalg.det(gam))
    v_l = gam @ v_u
    W = 1.0 / np.sqrt(1.0 - v_l @ v_u)
    u = np.concatenate([[W / alpha], W * (v_u - beta_u / alpha)])
    b0 = W * (B_u @ v_l) / alpha                       # Eq. 7a
    b = np.concatenate([[b0], (B_u + alpha * b0 * u[1:]) / W])   # Eq. 7b
    b2 = b @ g4 @ b
    if h is None:                                       # ideal gas; else the caller's specific enthalpy
        h = 1.0 + Gamma / (Gamma - 1.0) * P / rho
    T = (rho * h + b2) * np.outer(u, u) + (P + 0.5 * b2) * g4i - np.outer(b, b)   # Eq. 2
    Fd = np.outer(b, u) - np.outer(u, b)               # Eq. 3: (*F)^{mu nu}
    D = alpha * rho * u[0]
    T_ud = T @ g4                                       # T^mu_nu
    S = alpha * T_ud[0, 1:]
    tau = alpha ** 2 * T[0, 0] - D
    U = sg * np.concatenate([[D], S, [tau], B_u])
    F = np.zeros((3, 8))
    for j in range(3):
        F[j, 0] = alpha * rho * u[1 + j]
        F[j, 1:4] = alpha * T_ud[1 + j, 1:]
        F[j, 4] = alpha * (alpha * T[0, 1 + j] - rho * u[1 + j])
        F[j, 5:8] = alpha * Fd[1:, 1 + j]
    return U, sg * F, dict(W=W, h=h, b2=b2, sg=sg, T=T, g4=g4, alpha=alpha)


def slots(d):
    """map oracle 7-slot face flux (D,Sx,Sy,Sz,tau,Bt1,Bt2) -> indices into the 8-vector."""
    t1, t2 = (d + 1) % 3, (d + 2) % 3
    return [0, 1, 2, 3, 4, 5 + t1, 5 + t2]


def metric10(alpha, beta_u, g6):
    return np.concatenate([[alpha], beta_u, g6])
