"""Pins for the CPU fp64 oracle (oracle/tri_attn_oracle.c) -- SURVEY.md Sec. 8(c) pin table.

The paper prints no worked numeric example for EvoAttention (tests/golden/README.md), so the oracle
is pinned against what the mathematics fixes: an independent scalar brute force, closed forms,
invariants, central finite differences of L = sum(O*dO) (all five gradients, incl. dBias), and a
stock library routine (torch CPU fp64 softmax-attention + autograd).  Each test is chosen so that a
plausible slip (dropped term, wrong sign/index, transposed operand, scale on the bias) fails it.
"""
import itertools
import math

import numpy as np
import pytest

S, E = 0, 1


def T(x):
    """Swap the two N axes of an argument: [B,N,H,N,d] -> axes 1<->3; [B,H,N,N]/[B,N,N] -> last two."""
    if x is None:
        return None
    if x.ndim == 5:
        return np.ascontiguousarray(x.transpose(0, 3, 2, 1, 4))
    if x.ndim == 4 and x.shape[2] == x.shape[3] and x.shape[1] != x.shape[2]:
        return np.ascontiguousarray(x.transpose(0, 1, 3, 2))
    if x.ndim == 4:  # LSE [B,N,H,N]  or bias with H == N (ambiguous) -> caller must not rely on it
        raise ValueError("ambiguous 4-D transpose")
    if x.ndim == 3:
        return np.ascontiguousarray(x.transpose(0, 2, 1))
    raise ValueError


def T_bias(x):
    return np.ascontiguousarray(x.transpose(0, 1, 3, 2))


def T_lse(x):  # [B,N,H,N] -> swap axes 1 and 3
    return np.ascontiguousarray(x.transpose(0, 3, 2, 1))


def rand_problem(B, N, H, d, seed, mask_p=0.0, sigma_bias=1.0):
    r = np.random.default_rng(seed)
    shp = (B, N, H, N, d)
    p = {k: r.standard_normal(shp) for k in ("Q", "K", "V", "G", "dO")}
    p["bias"] = sigma_bias * r.standard_normal((B, H, N, N))
    if mask_p > 0:
        m = (r.random((B, N, N)) > mask_p).astype(np.uint8)
        # keep at least one key per (b, row) for both variants' readings
        for b in range(B):
            for x in range(N):
                m[b, x, x] = 1
        p["mask"] = m
    else:
        p["mask"] = None
    return p


# --------------------------------------------------------------------------------------------
# 1. Independent scalar brute force (pure Python, every index written out)
# --------------------------------------------------------------------------------------------
def brute_force(p, variant):
    Q, K, V, G, bias, mask, dO = (p[k] for k in ("Q", "K", "V", "G", "bias", "mask", "dO"))
    B, N, H, _, d = Q.shape
    O = np.zeros_like(Q)
    LSE = np.zeros((B, N, H, N))
    P = np.zeros((B, N, H, N, N))
    for b, i, h, j in itertools.product(range(B), range(N), range(H), range(N)):
        logits = []
        for k in range(N):
            if variant == S:
                kv, bb = K[b, i, h, k], bias[b, h, j, k]
                keep = True if mask is None else bool(mask[b, i, k])
            else:
                kv, bb = K[b, k, h, j], bias[b, h, k, i]
                keep = True if mask is None else bool(mask[b, k, j])
            s = sum(Q[b, i, h, j, c] * kv[c] for c in range(d)) / math.sqrt(d) + bb
            logits.append(s if keep else -math.inf)
        z = sum(math.exp(s) for s in logits)
        LSE[b, i, h, j] = math.log(z)
        for k in range(N):
            P[b, i, h, j, k] = math.exp(logits[k]) / z
        for c in range(d):
            a = 0.0
            for k in range(N):
                vv = V[b, i, h, k, c] if variant == S else V[b, k, h, j, c]
                a += P[b, i, h, j, k] * vv
            O[b, i, h, j, c] = a / (1.0 + math.exp(-G[b, i, h, j, c]))
    return O, LSE, P


@pytest.mark.parametrize("variant", [S, E])
@pytest.mark.parametrize("shape", [(1, 3, 1, 2), (2, 4, 2, 3)])
def test_forward_matches_scalar_brute_force(oracle, variant, shape):
    p = rand_problem(*shape, seed=11, mask_p=0.3)
    O, LSE, P = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], variant, return_P=True)
    Ob, Lb, Pb = brute_force(p, variant)
    np.testing.assert_allclose(O, Ob, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(LSE, Lb, rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(P, Pb, rtol=1e-12, atol=1e-14)


# --------------------------------------------------------------------------------------------
# 2. Softmax rows: sum to 1, >= 0, LSE = ln sum e^S
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [S, E])
def test_softmax_rows_sum_to_one(oracle, variant):
    p = rand_problem(2, 9, 3, 4, seed=3, mask_p=0.25, sigma_bias=3.0)
    O, LSE, P = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], variant, return_P=True)
    assert np.all(P >= 0)
    np.testing.assert_allclose(P.sum(-1), 1.0, atol=1e-14)
    # LSE against a direct numpy evaluation of the logits (starting only; ending via T below)
    if variant == S:
        Sx = np.einsum("bihjc,bihkc->bihjk", p["Q"], p["K"]) / math.sqrt(4) + p["bias"][:, None]
        Sx = np.where(p["mask"][:, :, None, None, :] > 0, Sx, -np.inf)
        np.testing.assert_allclose(LSE, np.log(np.exp(Sx).sum(-1)), rtol=1e-12)


# --------------------------------------------------------------------------------------------
# 3. Closed forms
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [S, E])
def test_zero_bias_identical_keys_gives_mean_of_values(oracle, variant):
    B, N, H, d = 1, 7, 2, 4
    p = rand_problem(B, N, H, d, seed=5)
    # identical keys along the key axis of the variant
    if variant == S:
        p["K"][:] = p["K"][:, :, :, :1, :]
        keep = np.ones((B, N, N), np.uint8)
        keep[:, :, -2:] = 0  # last two keys padded for every row
        meanV = p["V"][:, :, :, : N - 2, :].mean(3, keepdims=True)  # [B,i,H,1,d]
        meanV = np.broadcast_to(meanV, p["V"].shape)
    else:
        p["K"][:] = p["K"][:, :1]
        keep = np.ones((B, N, N), np.uint8)
        keep[:, -2:, :] = 0  # mask[b,k,j]
        meanV = np.broadcast_to(p["V"][:, : N - 2].mean(1, keepdims=True), p["V"].shape)
    bias = np.zeros((B, H, N, N))
    O, LSE = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], bias, keep, variant)
    np.testing.assert_allclose(O, meanV / (1 + np.exp(-p["G"])), rtol=1e-12, atol=1e-14)
    # LSE = s + ln(#unmasked) where s is the common logit
    if variant == S:
        s = np.einsum("bihjc,bihc->bihj", p["Q"], p["K"][:, :, :, 0]) / math.sqrt(d)
    else:
        s = np.einsum("bihjc,bhjc->bihj", p["Q"], p["K"][:, 0]) / math.sqrt(d)
    np.testing.assert_allclose(LSE, s + math.log(N - 2), rtol=1e-12)


def test_single_key_N1(oracle):
    p = rand_problem(2, 1, 3, 5, seed=8)
    for variant in (S, E):
        O, LSE = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], None, variant)
        np.testing.assert_allclose(O, p["V"] / (1 + np.exp(-p["G"])), rtol=1e-13)
        s = (p["Q"] * p["K"]).sum(-1) / math.sqrt(5) + p["bias"][:, :, 0, 0][:, None, :, None]
        np.testing.assert_allclose(LSE, s, rtol=1e-13)


def test_two_keys_is_logistic(oracle):
    """N=2: P[.,0] = logistic(s0 - s1) -- a textbook closed form with scale and bias visible."""
    p = rand_problem(1, 2, 1, 3, seed=21)
    _, _, P = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], None, S, return_P=True)
    for i, j in itertools.product(range(2), range(2)):
        s = [float(p["Q"][0, i, 0, j] @ p["K"][0, i, 0, k]) / math.sqrt(3) + p["bias"][0, 0, j, k]
             for k in range(2)]
        assert abs(P[0, i, 0, j, 0] - 1 / (1 + math.exp(s[1] - s[0]))) < 1e-14


def test_zero_queries_softmax_of_bias(oracle):
    p = rand_problem(1, 6, 2, 4, seed=9, mask_p=0.3)
    p["Q"][:] = 0
    _, _, P = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], S, return_P=True)
    Sx = np.where(p["mask"][:, :, None, None, :] > 0, p["bias"][:, None], -np.inf)  # [B,i,H,j,k]
    e = np.exp(Sx - Sx.max(-1, keepdims=True))
    np.testing.assert_allclose(P, e / e.sum(-1, keepdims=True), rtol=1e-13, atol=1e-15)


def test_convex_hull_and_open_gate(oracle):
    p = rand_problem(1, 8, 2, 4, seed=10)
    p["G"][:] = 50.0  # sigmoid -> 1
    O, _ = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], None, S)
    vmin = p["V"].min(3, keepdims=True)
    vmax = p["V"].max(3, keepdims=True)
    assert np.all(O >= vmin - 1e-12) and np.all(O <= vmax + 1e-12)


# --------------------------------------------------------------------------------------------
# 4. Bias / mask semantics
# --------------------------------------------------------------------------------------------
def test_bias_row_shift_and_permutations(oracle):
    B, N, H, d = 1, 6, 2, 4
    p = rand_problem(B, N, H, d, seed=12, mask_p=0.2)
    a = (p["Q"], p["K"], p["V"], p["G"])
    O, LSE = oracle.fwd(*a, p["bias"], p["mask"], S)
    dQ, dK, dV, dG, dB = oracle.bwd(p["dO"], *a, p["bias"], p["mask"], S)
    # (a) add c[b,h,j] to bias[b,h,j,:]: O unchanged, LSE shifts by c (scale must NOT touch bias)
    c = np.random.default_rng(1).standard_normal((B, H, N))
    O2, LSE2 = oracle.fwd(*a, p["bias"] + c[..., None], p["mask"], S)
    np.testing.assert_allclose(O2, O, rtol=1e-11, atol=1e-13)
    np.testing.assert_allclose(LSE2, LSE + c.transpose(0, 1, 2)[:, None], rtol=1e-12)
    # (b) permute keys: K,V rows; bias and mask columns -> O unchanged
    perm = np.random.default_rng(2).permutation(N)
    O3, _ = oracle.fwd(p["Q"], p["K"][:, :, :, perm], p["V"][:, :, :, perm], p["G"],
                       p["bias"][..., perm], p["mask"][..., perm], S)
    np.testing.assert_allclose(O3, O, rtol=1e-11, atol=1e-13)
    # (c) permute rows i: outputs permute, dBias unchanged
    rp = np.random.default_rng(3).permutation(N)
    a4 = tuple(x[:, rp] for x in a)
    O4, _ = oracle.fwd(*a4, p["bias"], p["mask"][:, rp], S)
    np.testing.assert_allclose(O4, O[:, rp], rtol=1e-12, atol=1e-14)
    dB4 = oracle.bwd(p["dO"][:, rp], *a4, p["bias"], p["mask"][:, rp], S)[4]
    np.testing.assert_allclose(dB4, dB, rtol=1e-10, atol=1e-13)


@pytest.mark.parametrize("variant", [S, E])
def test_masked_keys_get_exact_zeros(oracle, variant):
    B, N, H, d = 2, 7, 2, 3
    p = rand_problem(B, N, H, d, seed=13)
    keep = np.ones((B, N), np.uint8)
    keep[0, [1, 4]] = 0
    keep[1, [6]] = 0
    mask = (np.broadcast_to(keep[:, None, :], (B, N, N)) if variant == S
            else np.broadcast_to(keep[:, :, None], (B, N, N))).copy()
    _, _, P = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], mask, variant, return_P=True)
    dQ, dK, dV, dG, dB = oracle.bwd(p["dO"], p["Q"], p["K"], p["V"], p["G"], p["bias"], mask, variant)
    for b in range(B):
        for k in np.where(keep[b] == 0)[0]:
            assert np.all(P[b, ..., k] == 0)
            if variant == S:
                assert np.all(dK[b, :, :, k] == 0) and np.all(dV[b, :, :, k] == 0)
                assert np.all(dB[b, :, :, k] == 0)
            else:
                assert np.all(dK[b, k] == 0) and np.all(dV[b, k] == 0)
                assert np.all(dB[b, :, k, :] == 0)


def test_fully_masked_row_convention(oracle):
    """Reading A6: a row with every key masked gives P=0, O=0, LSE=-inf, zero gradients."""
    B, N, H, d = 1, 5, 2, 3
    p = rand_problem(B, N, H, d, seed=14)
    mask = np.ones((B, N, N), np.uint8)
    mask[0, 2, :] = 0  # row i=2 has no visible key (starting)
    O, LSE, P = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], mask, S, return_P=True)
    assert np.all(O[0, 2] == 0) and np.all(np.isneginf(LSE[0, 2])) and np.all(P[0, 2] == 0)
    g = oracle.bwd(p["dO"], p["Q"], p["K"], p["V"], p["G"], p["bias"], mask, S)
    for x in g[:4]:
        assert np.all(x[0, 2] == 0) and np.all(np.isfinite(x))
    assert np.all(np.isfinite(g[4]))


# --------------------------------------------------------------------------------------------
# 5. Backward: finite differences of L = sum(O * dO), every input incl. bias
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [S, E])
def test_backward_matches_central_finite_differences(oracle, variant):
    B, N, H, d = 2, 4, 2, 3
    p = rand_problem(B, N, H, d, seed=17 + variant, mask_p=0.25)
    names = ("Q", "K", "V", "G", "bias")
    grads = dict(zip(names, oracle.bwd(p["dO"], p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], variant)))

    def loss(q):
        O, _ = oracle.fwd(q["Q"], q["K"], q["V"], q["G"], q["bias"], p["mask"], variant)
        return float((O * p["dO"]).sum())

    eps = 1e-6
    rng = np.random.default_rng(0)
    for name in names:
        x = p[name]
        idxs = [tuple(rng.integers(0, s) for s in x.shape) for _ in range(40)]
        if x.size <= 200:
            idxs = list(np.ndindex(*x.shape))
        for idx in idxs:
            old = x[idx]
            x[idx] = old + eps
            lp = loss(p)
            x[idx] = old - eps
            lm = loss(p)
            x[idx] = old
            fd = (lp - lm) / (2 * eps)
            an = grads[name][idx]
            assert abs(fd - an) <= 1e-6 * max(1.0, abs(an)) + 2e-8, (name, idx, fd, an)


@pytest.mark.parametrize("variant", [S, E])
def test_backward_identities(oracle, variant):
    B, N, H, d = 2, 8, 2, 4
    p = rand_problem(B, N, H, d, seed=23, mask_p=0.2)
    a = (p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"])
    O, LSE, P = oracle.fwd(*a, variant, return_P=True)
    dQ, dK, dV, dG, dB = oracle.bwd(p["dO"], *a, variant)
    sg = 1 / (1 + np.exp(-p["G"]))
    # dG = dO (.) O (.) (1 - sg)   (reading A3)
    np.testing.assert_allclose(dG, p["dO"] * O * (1 - sg), rtol=1e-11, atol=1e-14)
    # sum_k dS = 0  =>  rows of dBias along the key axis sum to 0
    key_axis = 3 if variant == S else 2
    np.testing.assert_allclose(dB.sum(key_axis), 0.0, atol=1e-12)
    # sum_k P dP = rowsum(dO (.) O)   (the shortcut of P:L437 / P:L511 with the gated O)
    dA = p["dO"] * sg
    if variant == S:
        dP = np.einsum("bihjc,bihkc->bihjk", dA, p["V"])
    else:
        dP = np.einsum("bihjc,bkhjc->bihjk", dA, p["V"])
    np.testing.assert_allclose((P * dP).sum(-1), (p["dO"] * O).sum(-1), rtol=1e-11, atol=1e-13)
    # dBias equals the explicit sum of dS over the broadcast axis
    dS = P * (dP - (P * dP).sum(-1, keepdims=True))
    ref = dS.sum(1) if variant == S else dS.sum(3).transpose(0, 2, 3, 1)  # -> [b,h,k,i]
    np.testing.assert_allclose(dB, ref, rtol=1e-11, atol=1e-13)


# --------------------------------------------------------------------------------------------
# 6. Ending node == T . starting . T  (ending coded directly from its index formulas)
# --------------------------------------------------------------------------------------------
def test_ending_equals_transposed_starting(oracle):
    B, N, H, d = 2, 6, 3, 4
    p = rand_problem(B, N, H, d, seed=31, mask_p=0.2)
    Oe, LSEe = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], E)
    ge = oracle.bwd(p["dO"], p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], E)
    tq, tk, tv, tg, tdo = (T(p[k]) for k in ("Q", "K", "V", "G", "dO"))
    tb, tm = T_bias(p["bias"]), T(p["mask"])
    Os, LSEs = oracle.fwd(tq, tk, tv, tg, tb, tm, S)
    gs = oracle.bwd(tdo, tq, tk, tv, tg, tb, tm, S)
    np.testing.assert_allclose(Oe, T(Os), rtol=1e-12, atol=1e-14)
    np.testing.assert_allclose(LSEe, T_lse(LSEs), rtol=1e-12)
    for x, y in zip(ge[:4], gs[:4]):
        np.testing.assert_allclose(x, T(y), rtol=1e-11, atol=1e-14)
    np.testing.assert_allclose(ge[4], T_bias(gs[4]), rtol=1e-11, atol=1e-14)


# --------------------------------------------------------------------------------------------
# 7. Library cross-check: torch CPU fp64 softmax attention + autograd
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("variant", [S, E])
def test_against_torch_fp64_sdpa_autograd(oracle, variant):
    torch = pytest.importorskip("torch")
    B, N, H, d = 2, 10, 3, 8
    p = rand_problem(B, N, H, d, seed=41, mask_p=0.2, sigma_bias=2.0)
    tt = {k: torch.tensor(p[k], dtype=torch.float64, requires_grad=True) for k in ("Q", "K", "V", "G", "bias")}
    mask = torch.tensor(p["mask"]).bool()
    if variant == S:
        q, k, v = tt["Q"], tt["K"], tt["V"]  # [B,i,H,n,d]
        add = tt["bias"][:, None] + torch.where(mask, 0.0, -math.inf)[:, :, None, None, :].double()
        a = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=add)
    else:
        q, k, v = (tt[n].permute(0, 3, 2, 1, 4) for n in ("Q", "K", "V"))  # [B,j,H,n,d]
        # bias[b,h,k,i] -> [b,1,h,i,k]; mask[b,k,j] -> [b,j,1,1,k]
        add = tt["bias"].transpose(2, 3)[:, None] + \
            torch.where(mask, 0.0, -math.inf).double().permute(0, 2, 1)[:, :, None, None, :]
        a = torch.nn.functional.scaled_dot_product_attention(q, k, v, attn_mask=add).permute(0, 3, 2, 1, 4)
    O_t = torch.sigmoid(tt["G"]) * a
    (O_t * torch.tensor(p["dO"])).sum().backward()
    O, _ = oracle.fwd(p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], variant)
    g = oracle.bwd(p["dO"], p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"], variant)
    np.testing.assert_allclose(O, O_t.detach().numpy(), rtol=1e-10, atol=1e-12)
    for name, x in zip(("Q", "K", "V", "G", "bias"), g):
        np.testing.assert_allclose(x, tt[name].grad.numpy(), rtol=1e-9, atol=1e-12, err_msg=name)


# --------------------------------------------------------------------------------------------
# 8. Decoupled shapes (used by the full-size sampled parity checks) reduce to the square operator
# --------------------------------------------------------------------------------------------
def test_general_shape_core_is_consistent_with_square(oracle):
    B, N, H, d = 1, 7, 2, 4
    p = rand_problem(B, N, H, d, seed=51, mask_p=0.2)
    a = (p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"])
    O, LSE = oracle.fwd(*a, S)
    dQ, dK, dV, dG, dB = oracle.bwd(p["dO"], *a, S)
    rows = [1, 4]
    Os, Ls = oracle.fwd_start_general(p["Q"][:, rows], p["K"][:, rows], p["V"][:, rows], p["G"][:, rows],
                                      p["bias"], p["mask"][:, rows])
    np.testing.assert_array_equal(Os, O[:, rows])
    np.testing.assert_array_equal(Ls, LSE[:, rows])
    gs = oracle.bwd_start_general(p["dO"][:, rows], p["Q"][:, rows], p["K"][:, rows], p["V"][:, rows],
                                  p["G"][:, rows], p["bias"], p["mask"][:, rows])
    for x, y in zip(gs[:4], (dQ, dK, dV, dG)):
        np.testing.assert_array_equal(x, y[:, rows])
    qs = [0, 3, 6]  # query subset: O, LSE, dQ, dG, dBias rows are exact
    Oq, Lq = oracle.fwd_start_general(p["Q"][:, :, :, qs], p["K"], p["V"], p["G"][:, :, :, qs],
                                      p["bias"][:, :, qs], p["mask"])
    np.testing.assert_array_equal(Oq, O[:, :, :, qs])
    gq = oracle.bwd_start_general(p["dO"][:, :, :, qs], p["Q"][:, :, :, qs], p["K"], p["V"],
                                  p["G"][:, :, :, qs], p["bias"][:, :, qs], p["mask"])
    np.testing.assert_array_equal(gq[0], dQ[:, :, :, qs])
    np.testing.assert_array_equal(gq[3], dG[:, :, :, qs])
    np.testing.assert_array_equal(gq[4], dB[:, :, qs])


def test_general_shape_dbias_is_additive_over_row_partitions_and_rows_may_exceed_n(oracle):
    """What the row-chunked host pipeline, the EvoSP row shards and the R != N entry points rely on: with the bias plane
    fixed, the rows are independent problems, so dBias of a row set is the sum of the dBias of any partition of it (here
    against the square problem's dBias), a single row (R = 1) is a legal problem, and R may exceed N (rows of two unrelated
    draws stacked: every per-row output equals that of the problem the row came from)."""
    B, N, H, d = 1, 6, 2, 4
    p = rand_problem(B, N, H, d, seed=61, mask_p=0.25)
    q = rand_problem(B, N, H, d, seed=62, mask_p=0.25)
    a = (p["Q"], p["K"], p["V"], p["G"], p["bias"], p["mask"])
    dB_all = oracle.bwd(p["dO"], *a, S)[4]
    parts = ([0], [1, 2, 3], [4, 5])
    acc = np.zeros_like(dB_all)
    for rows in parts:
        acc += oracle.bwd_start_general(p["dO"][:, rows], p["Q"][:, rows], p["K"][:, rows], p["V"][:, rows], p["G"][:, rows],
                                        p["bias"], p["mask"][:, rows])[4]
    np.testing.assert_allclose(acc, dB_all, rtol=1e-13, atol=1e-14)
    # R = 2 N rows: p's rows followed by q's rows, all under p's bias
    cat = {k: np.concatenate([p[k], q[k]], axis=1) for k in ("Q", "K", "V", "G", "dO", "mask")}
    O2, L2 = oracle.fwd_start_general(cat["Q"], cat["K"], cat["V"], cat["G"], p["bias"], cat["mask"])
    g2 = oracle.bwd_start_general(cat["dO"], cat["Q"], cat["K"], cat["V"], cat["G"], p["bias"], cat["mask"])
    Op, Lp = oracle.fwd(*a, S)
    Oq, Lq = oracle.fwd_start_general(q["Q"], q["K"], q["V"], q["G"], p["bias"], q["mask"])
    np.testing.assert_array_equal(O2[:, :N], Op)
    np.testing.assert_array_equal(O2[:, N:], Oq)
    np.testing.assert_array_equal(L2[:, :N], Lp)
    gq = oracle.bwd_start_general(q["dO"], q["Q"], q["K"], q["V"], q["G"], p["bias"], q["mask"])
    np.testing.assert_array_equal(g2[0][:, N:], gq[0])
    np.testing.assert_allclose(g2[4], dB_all + gq[4], rtol=1e-13, atol=1e-14)
