"""Independent dense numpy evaluation of the GFN-style network (test helper).

Written separately from oracle/pimd_oracle.c and in a DIFFERENT algebraic form: the running-sum
form e^l_ij = e^0_ij + E^l_i + E^l_j on dense (N, N) arrays, whereas the oracle
stores and updates a per-pair edge state literally as in PAPER.md L74.  Agreement of the two pins
both the oracle's indexing and the G5 identity the CUDA path relies on.
"""
import numpy as np


def unpack(w, S, K, H, L):
    w = np.asarray(w, dtype=np.float64)
    o = [0]

    def take(*shape):
        n = int(np.prod(shape))
        a = w[o[0]:o[0] + n].reshape(shape)
        o[0] += n
        return a

    d = {"Emb": take(S, H), "W_e1": take(H, K), "b_e1": take(H), "W_e2": take(H, H), "b_e2": take(H), "layers": []}
    for _ in range(L):
        d["layers"].append({"W_s": take(H, H), "W_vn": take(H, H), "W_vm": take(H, H), "b_v1": take(H),
                            "W_v2": take(H, H), "b_v2": take(H), "W_a": take(H, H), "b_a": take(H)})
    d.update({"W_f1": take(H, H), "b_f1": take(H), "w_f2": take(H), "b_f2": take(1)[0]})
    assert o[0] == w.size
    return d


def silu(x):
    return x / (1.0 + np.exp(-x))


def dense_forces(species, x, box, w, S, K, H, L, r_cut, agg_norm, force_scale, gross=False):
    """x [N,3]; box [3] (zeros = open).  Returns F [N,3]; with gross=True also the sum of the
    magnitudes of all terms of F_i, force_scale * sum_j c_ij (sum_o |w_f2[o] SiLU(t_o)| + |b_f2|)  [N]."""
    p = unpack(w, S, K, H, L)
    N = x.shape[0]
    delta = x[None, :, :] - x[:, None, :]  # delta[i, j] = x_j - x_i
    if box[0] > 0:
        t = delta / box
        delta = delta - box * (np.sign(t) * np.floor(np.abs(t) + 0.5))
    d = np.sqrt((delta ** 2).sum(-1))
    mask = ((delta ** 2).sum(-1) < r_cut * r_cut) & ~np.eye(N, dtype=bool)
    dd = np.where(mask, d, 1.0)
    u = -delta / dd[..., None]
    c = np.where(mask, 0.5 * (np.cos(np.pi * d / r_cut) + 1.0), 0.0)
    dl = r_cut / (K - 1)
    g = np.exp(-((d[..., None] - dl * np.arange(K)) ** 2) / (2 * dl * dl))  # [N,N,K]
    e0 = silu(g @ p["W_e1"].T + p["b_e1"]) @ p["W_e2"].T + p["b_e2"]  # [N,N,H]
    n = p["Emb"][species]
    E = np.zeros((N, H))
    for lay in p["layers"]:
        xs = n @ lay["W_s"].T
        e = e0 + E[:, None, :] + E[None, :, :]
        m = agg_norm * np.einsum("ij,ijh,jh->ih", c, e, xs)
        n = n + silu(n @ lay["W_vn"].T + m @ lay["W_vm"].T + lay["b_v1"]) @ lay["W_v2"].T + lay["b_v2"]
        E = E + n @ lay["W_a"].T + lay["b_a"]
    e = e0 + E[:, None, :] + E[None, :, :]
    act = silu(e @ p["W_f1"].T + p["b_f1"])
    s = act @ p["w_f2"] + p["b_f2"]  # [N,N]
    F = force_scale * np.einsum("ij,ij,ija->ia", c, s, u)
    if gross:
        return F, abs(force_scale) * (c * (np.abs(act) @ np.abs(p["w_f2"]) + abs(p["b_f2"]))).sum(axis=1)
    return F
