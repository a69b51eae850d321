"""Seeded synthetic inputs and layout marshalling shared by the oracle tests and the GPU parity
tests.  Holds none of the method's arithmetic: only numpy random draws, Lorentz transformations of
test momenta and AoS <-> SoA reshapes."""
import numpy as np


def random_lorentz(seed):
    """A proper orthochronous Lorentz matrix: random rotation times a random boost (|beta| < 0.8)."""
    rng = np.random.default_rng(seed)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    rot = np.eye(4)
    rot[1:, 1:] = q
    beta = rng.normal(size=3)
    beta *= rng.uniform(0.1, 0.8) / np.linalg.norm(beta)
    b2 = beta @ beta
    g = 1.0 / np.sqrt(1.0 - b2)
    boost = np.eye(4)
    boost[0, 0] = g
    boost[0, 1:] = g * beta
    boost[1:, 0] = g * beta
    boost[1:, 1:] += (g - 1.0) * np.outer(beta, beta) / b2
    return boost @ rot


def transform(mom, lam):
    """mom[n, npar, 4] -> Lambda applied to every 4-vector."""
    return np.einsum("ab,npb->npa", lam, mom)


def aos_to_soa(a):
    """[n, k, 4] event-major -> [k*4, n] component-major with the event index fastest (include/mg.h layout)."""
    n = a.shape[0]
    return np.ascontiguousarray(a.reshape(n, -1).T)


def soa_to_aos(a, k):
    """[k*4, n] -> [n, k, 4]."""
    return np.ascontiguousarray(a.T).reshape(a.shape[1], k, 4)


def read_worked_examples(path):
    out = []
    cur = None
    for line in open(path):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        t = line.split()
        if t[0] == "process":
            cur = {"process": int(t[1]), "me": float(t[3]), "mom": []}
            out.append(cur)
        else:
            cur["mom"].append([float(x) for x in t])
    for c in out:
        c["mom"] = np.array(c["mom"])[None]
    return out
