"""fp64 numpy evaluation of the GFN-style network with selected operands rounded to bf16 (test helper).

Purpose: derive, from arithmetic alone, the force error that `gemm_dtype = 1` (BASELINE.json configs[3..4]:
"bf16 atom-wise GEMMs and fp32 accumulation") introduces, so that the tolerance the CUDA path is held to
 is pinned by the operand precision and not by where a kernel happens to land.
Everything is computed in fp64; a quantity in `rounding` (a set of keys, or
a dict key -> rounding function) is passed through round-to-nearest-even bf16 (8 significand bits), or the given
function, at the point where the tcgen05 path stores it as a GEMM operand:

    'rbf'   Gaussian basis g(d) and W_e1                    (first filter product)
    'h1'    h1 = SiLU(W_e1 g + b), W_e2 and W_f1 W_e2       (second filter product, message and head)
    'x'     x_j = W_s n_j as gathered by the message pass   (operand of the pair-index contraction)
    'E'     the running edge sums E_i, E_j                  (NOT a GEMM operand: kept fp32 by the product path)
    'node'  n, m, SiLU(.) and the atom-wise weights         (atom-wise GEMM operands)
    'G'     G = W_f1 E as gathered by the head              (NOT a GEMM operand)
    'act'   SiLU(W_fe h1 + b + G_i + G_j) and w_f2          (readout product of the head)

Independent of oracle/ and of the CUDA path; shares only `dense_gfn.unpack/silu` (tests/).
"""
import numpy as np

from dense_gfn import unpack, silu

GEMM_OPERANDS = frozenset({"rbf", "h1", "x", "node", "act"})   # what configs[3..4] allow to be bf16
ALL = frozenset({"rbf", "h1", "x", "E", "node", "G", "act"})


def bf16(a):
    """round-to-nearest-even to bfloat16, returned as fp64"""
    a = np.asarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).astype(np.float64)


def bf16x2(a):
    """a bf16 pair hi + lo (hi = bf16(v), lo = bf16(v - hi)): what the split-precision atom-wise products carry"""
    a32 = np.asarray(a, dtype=np.float32).astype(np.float64)
    hi = bf16(a32)
    return hi + bf16(a32 - hi)


def f16(a):
    """IEEE binary16 (the head's readout operand)"""
    return np.asarray(a, dtype=np.float32).astype(np.float16).astype(np.float64)


# what the tcgen05 path of paper_2503_23728_b200 rounds, and how (gfn_pair_pipe.cu, gfn_node_tc.cu): G stays fp32
PRODUCT_PATH = {"rbf": bf16, "h1": bf16, "x": bf16, "E": bf16, "node": bf16x2, "act": f16}


def dense_forces_rounded(species, x, box, w, S, K, H, L, r_cut, agg_norm, force_scale, rounding=GEMM_OPERANDS):
    """x [N,3]; box [3] (zeros = open).  Returns F [N,3] (fp64 arithmetic, bf16-rounded operands)."""
    if not isinstance(rounding, dict):
        rounding = {k: bf16 for k in rounding}
    r = lambda a, key: rounding[key](a) if key in rounding else a
    p = unpack(w, S, K, H, L)
    N = x.shape[0]
    delta = x[None, :, :] - x[:, None, :]
    if box[0] > 0:
        t = delta / box
        delta = delta - box * (np.sign(t) * np.floor(np.abs(t) + 0.5))
    d2 = (delta ** 2).sum(-1)
    d = np.sqrt(d2)
    mask = (d2 < r_cut * r_cut) & ~np.eye(N, dtype=bool)
    u = -delta / np.where(mask, d, 1.0)[..., None]
    c = np.where(mask, 0.5 * (np.cos(np.pi * d / r_cut) + 1.0), 0.0)
    dl = r_cut / (K - 1)
    g = np.exp(-((d[..., None] - dl * np.arange(K)) ** 2) / (2 * dl * dl))
    h1 = r(silu(r(g, "rbf") @ r(p["W_e1"], "rbf").T + p["b_e1"]), "h1")
    e0 = h1 @ r(p["W_e2"], "h1").T + p["b_e2"]
    n = p["Emb"][species]
    E = np.zeros((N, H))
    xs = n @ p["layers"][0]["W_s"].T if L > 0 else None      # layer 0: one exact vector per species
    for li, lay in enumerate(p["layers"]):
        Eg = r(E, "E")
        e = e0 + Eg[:, None, :] + Eg[None, :, :]
        m = agg_norm * np.einsum("ij,ijh,jh->ih", c, e, r(xs, "x"))
        hid = silu(r(n, "node") @ r(lay["W_vn"], "node").T + r(m, "node") @ r(lay["W_vm"], "node").T + lay["b_v1"])
        n = n + r(hid, "node") @ r(lay["W_v2"], "node").T + lay["b_v2"]
        E = E + r(n, "node") @ r(lay["W_a"], "node").T + lay["b_a"]
        if li + 1 < L:
            xs = r(n, "node") @ r(p["layers"][li + 1]["W_s"], "node").T
    G = r(r(E, "node") @ r(p["W_f1"], "node").T if L > 0 else np.zeros((N, H)), "G")
    Wfe = p["W_f1"] @ p["W_e2"]
    bfe = p["W_f1"] @ p["b_e2"] + p["b_f1"]
    t = h1 @ r(Wfe, "h1").T + bfe + G[:, None, :] + G[None, :, :]
    s = r(silu(t), "act") @ r(p["w_f2"], "act") + p["b_f2"]
    return force_scale * np.einsum("ij,ij,ija->ia", c, s, u)


def spec_form_error(F, Fref):
    """The north-star tolerance in a well-defined relative form: per atom
    |dF_i|_2 / max(|F_i|_2, rms_i |F_i|_2).  Returns (max over atoms, rms|dF| / rms|F|)."""
    dn = np.linalg.norm(F - Fref, axis=-1)
    fn = np.linalg.norm(Fref, axis=-1)
    rms = np.sqrt((fn ** 2).mean())
    return float((dn / np.maximum(fn, rms)).max()), float(np.sqrt((dn ** 2).mean()) / rms)
