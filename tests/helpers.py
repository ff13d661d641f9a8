"""Shared test helpers (no method arithmetic beyond plain reconstruction)."""
import numpy as np


def mask_of(n):
    return np.uint64((1 << n) - 1) if n < 64 else np.uint64(0xFFFFFFFFFFFFFFFF)


def pack_bits(z):
    """z: uint8 [n_bits, count] -> uint64 words with bit j = z[j]."""
    w = np.zeros(z.shape[1], np.uint64)
    for j in range(z.shape[0]):
        w |= z[j].astype(np.uint64) << np.uint64(j)
    return w


def all_r_keys(P, n, seed, r_out=None):
    """One element per mask value r = 0..2^n-1 (keys depend on r only, so each x reuses them)."""
    N = 1 << n
    r_in = np.arange(N, dtype=np.uint64)
    return r_in, P.keygen(r_in, r_out, seed)


def random_spec(seed, variant=0):
    """A random well-formed operator specification + Phi program (Def 4.1 / 4.2 grammar) for differential testing of
    the two independent compilers and of the CUDA path against the oracle.  Holds no method arithmetic."""
    from workloads import specs as S
    rng = np.random.default_rng(seed)
    n = int(rng.choice([8, 12, 16, 33, 64]))
    N = 1 << n
    f = int(rng.integers(1, min(n, 13)))
    m = int(rng.integers(1, 7))
    r = int(rng.integers(1, 3))
    d = int(rng.integers(0, 3))
    p_aux = int(rng.integers(0, 2)) if r * (d + 1) < 8 else 0
    cuts = sorted({int(v) for v in rng.integers(1, N, size=m - 1, dtype=np.uint64)} | ({N // 2} if m > 1 and rng.random() < 0.5 else set()))
    m = len(cuts) + 1
    R = lambda: int(rng.integers(0, 1 << 63, dtype=np.uint64)) * 2 + int(rng.integers(0, 2))
    coeff = [[[R() if rng.random() < 0.8 else 0 for _ in range(d + 1)] for _ in range(r)] for _ in range(m)]
    aux = [[R() for _ in range(p_aux)] for _ in range(m)]
    nodes = []
    for i in range(int(rng.integers(1, 9))):
        kind = int(rng.choice([S.BN_CONST, S.BN_C, S.BN_D, S.BN_MSB, S.BN_CARRY] if i < 2 else
                              [S.BN_C, S.BN_D, S.BN_MSB, S.BN_CARRY, S.BN_NOT, S.BN_XOR, S.BN_AND, S.BN_OR, S.BN_XOR]))
        k = int(rng.integers(1, n + 1)) if kind in (S.BN_D, S.BN_CARRY) else 0
        lhs = int(rng.integers(0, i)) if kind >= S.BN_NOT else 0
        rhs = int(rng.integers(0, i)) if kind >= S.BN_XOR else 0
        is2k = int(kind in (S.BN_C, S.BN_D) and rng.random() < 0.1)
        lim = (1 << k) if kind == S.BN_D else N
        value = 0 if is2k else (int(rng.integers(0, lim, dtype=np.uint64)) if kind in (S.BN_C, S.BN_D, S.BN_MSB) else int(rng.integers(0, 2)))
        nodes.append((kind, k, lhs, rhs, is2k, value))
    ell = int(rng.integers(0, 4))
    uniform = rng.random() < 0.5
    base = [int(rng.integers(0, len(nodes))) for _ in range(ell)]
    bit_root = [base if uniform else [int(rng.integers(0, len(nodes))) for _ in range(ell)] for _ in range(m)]
    kappa_a = [(S.KA_R_SHR, int(rng.integers(0, n)))] if rng.random() < 0.5 else []
    kappa_b = [(S.KB_R_BIT, int(rng.integers(0, n)))] if rng.random() < 0.5 else []
    phi, n_out_a, n_out_b = [], r, ell
    if rng.random() < 0.7:
        A, B = [], []                                               # defined registers
        def newA(op, a=0, b=0, imm=0):
            phi.append((op, len(A), a, b, imm)); A.append(len(A)); return len(A) - 1
        def newB(op, a=0, b=0, imm=0):
            phi.append((op, len(B), a, b, imm)); B.append(len(B)); return len(B) - 1
        newA(S.PHI_A_X)
        for j in range(r):
            newA(S.PHI_A_Y, j)
        for j in range(p_aux):
            newA(S.PHI_A_AUX, j)
        if kappa_a:
            newA(S.PHI_A_KAPPA, 0)
        newA(S.PHI_A_CONST, imm=R() & (N - 1))
        newA(S.PHI_A_XHAT_SHR, int(rng.integers(0, n)))
        for j in range(ell):
            newB(S.PHI_B_Z, j)
        if kappa_b:
            newB(S.PHI_B_KAPPA, 0)
        newB(S.PHI_B_XHAT, int(rng.integers(0, n)))
        newB(S.PHI_B_CONST, imm=int(rng.integers(0, 2)))
        for _ in range(int(rng.integers(2, 9))):
            if rng.random() < 0.55:
                op = int(rng.choice([S.PHI_A_ADD, S.PHI_A_SUB, S.PHI_A_MULC, S.PHI_A_MUL, S.PHI_A_B2A]))
                if op == S.PHI_A_B2A:
                    newA(op, int(rng.choice(B)))
                else:
                    newA(op, int(rng.choice(A)), int(rng.choice(A)), R() & (N - 1))
            else:
                op = int(rng.choice([S.PHI_B_NOT, S.PHI_B_XOR, S.PHI_B_AND, S.PHI_B_OR, S.PHI_B_ANDPUB]))
                if op == S.PHI_B_ANDPUB:
                    newB(op, int(rng.choice(B)), int(rng.integers(0, n)), int(rng.integers(0, 2)))
                else:
                    newB(op, int(rng.choice(B)), int(rng.choice(B)))
        rng_a2b = np.random.default_rng(seed + 7777)                # A2B nodes (own stream: the rest of the spec is as before)
        for _ in range(int(rng_a2b.integers(0, 3))):
            newB(S.PHI_B_A2B, int(rng_a2b.choice(A)), int(rng_a2b.integers(0, n)))
            if rng_a2b.random() < 0.5:
                newA(S.PHI_A_B2A, B[-1])                             # and back into arithmetic
        n_out_a, n_out_b = int(rng.integers(1, 3)), int(rng.integers(0, 4))
        for j in range(n_out_a):
            phi.append((S.PHI_A_OUT, j, int(rng.choice(A)), 0, 0))
        for j in range(n_out_b):
            phi.append((S.PHI_B_OUT, j, int(rng.choice(B)), 0, 0))
    spec = S._mk(f"rand{seed}_n{n}", n, f, cuts, coeff, nodes=nodes, bit_root=bit_root if ell else None, aux=aux if p_aux else None,
                 kappa_a=kappa_a, kappa_b=kappa_b, phi=phi, n_out_a=n_out_a, n_out_b=n_out_b,
                 mask_output=bool(rng.random() < 0.3), out_frac=f)
    spec.variant = variant if (not (variant & 4) or d <= 2) else variant & ~4
    return spec


# ---- brute-force harness shared by test_oracle_gate.py / test_oracle_sp.py ------------------------------------------
_PMAP_JOB = None        # (fn, items) of the running pmap: forked workers inherit it, so closures need no pickling


def _pmap_call(i):
    fn, items = _PMAP_JOB
    return fn(items[i])


def pmap(fn, items, workers=None, threads=False):
    """Run fn over items on all host cores (threads=True: a thread pool -- for callers that hold a CUDA context, which must not
    be forked).  The oracle is plain single-threaded C behind ctypes and keeps no mutable global
    state after orc_compile() (its AES tables are filled there), so independent calls can run side by side; this is what makes
    the exhaustive pins affordable -- the oracle's arithmetic itself stays single-threaded.  Workers are FORKED processes (they
    inherit the compiled program and the closure; the numpy checks around each oracle call would serialise threads on the GIL);
    where fork is unavailable, a thread pool (ctypes releases the GIL during the C calls).  Exceptions (assertion failures)
    propagate; results come back in order."""
    global _PMAP_JOB
    import multiprocessing as mp
    import os
    items = list(items)
    workers = workers or min(len(items), os.cpu_count() or 1)
    if workers <= 1 or _PMAP_JOB is not None:                  # serial, or already inside a worker
        return [fn(it) for it in items]
    if not threads and "fork" in mp.get_all_start_methods():
        _PMAP_JOB = (fn, items)
        import warnings
        try:
            with warnings.catch_warnings():
                # the parent may hold idle library threads (BLAS, torch); the workers only call the oracle's C and element-wise numpy
                warnings.filterwarnings("ignore", message=".*multi-threaded, use of fork.*", category=DeprecationWarning)
                with mp.get_context("fork").Pool(workers) as pool:
                    return pool.map(_pmap_call, range(len(items)), chunksize=max(1, len(items) // (4 * workers)))
        finally:
            _PMAP_JOB = None
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=workers) as ex:
        return list(ex.map(fn, items))


def expected_atoms(P, x, r_in, n):
    """The T bits the packed comparison must reconstruct to, from their plain definitions (Def I.1).
    Protocol-3 construction: atom t = I[view_{k,c}(xhat) < theta_t], theta_t = (r_k + beta_t) mod 2^k (r-atom: r_k).
    Single-key construction (variant bit 0): a theta-atom IS the predicate I[view_{k,c}(x) < beta_t]; r-atoms as above."""
    xhat = (x + r_in) & mask_of(n)
    sp = bool(getattr(P.spec, "variant", 0) & 1)
    rows = []
    for t in range(P.shape["T"]):
        a = P.atom(t)
        K = np.uint64((1 << a["k"]) - 1) if a["k"] < 64 else np.uint64(0xFFFFFFFFFFFFFFFF)
        u = ((xhat & K) + np.uint64(a["c"])) & K
        rk = r_in & K
        if not a["is_theta"]:
            rows.append(u < rk)
        elif sp:
            rows.append((((x & K) + np.uint64(a["c"])) & K) < np.uint64(a["beta"]))
        else:
            rows.append(u < ((rk + np.uint64(a["beta"])) & K))
    return rows


def check_gate_outputs(P, spec, x, r_in, r_out, out, calls=True):
    """Lemma 4.5 / Thm 4.6: the two parties' outputs reconstruct to the plaintext G(x) (Tier A), and
    (calls=True) each of the two FSS calls reconstructs to its plain definition: Def I.1 bits, Def I.2 = the payload of
    the interval that contains x.  x, r_in: arrays of the same length; r_out: [n_out_a, count] or None."""
    n = spec.n
    M = mask_of(n)
    ye, ze = P.plain_G(x, r_in)
    if spec.mask_output:
        ye = (ye + r_out[: ye.shape[0]]) & M
    assert np.array_equal((out["y"][0] + out["y"][1]) & M, ye), (spec.name, "y")
    if P.shape["n_out_b"]:
        assert np.array_equal(out["z"][0] ^ out["z"][1], pack_bits(ze)), (spec.name, "z")
    if not calls:
        return
    word = out["bits"][0] ^ out["bits"][1]
    for t, want in enumerate(expected_atoms(P, x, r_in, n)):
        got = (word >> np.uint64(t)) & np.uint64(1)
        assert np.array_equal(got, want.astype(np.uint64)), (spec.name, "atom", t)
    if P.shape["has_lut"] and not (getattr(spec, "variant", 0) & 4):
        c = (out["coeff"][0] + out["coeff"][1]) & M
        i_star = np.searchsorted(np.array([0] + spec.alpha, dtype=np.uint64), x, side="right") - 1
        pay = np.concatenate([spec.coeff.reshape(spec.m, -1), spec.aux.reshape(spec.m, -1)], axis=1) & M
        assert np.array_equal(c, pay[i_star].T), (spec.name, "lookup")


def r_out_for(P, n, count):
    na = max(1, P.shape["n_out_a"])
    return ((np.arange(count * na, dtype=np.uint64) * np.uint64(2654435761)) & mask_of(n)).reshape(na, count)


def check_all_r(orc, spec, xs, seed=11, calls=True):
    """Every mask r in Z_{2^n} (both Protocol 3 branches) for each x in xs.  The keys depend on r only, so they
    are generated once (in parallel chunks: the dealer's randomness is indexed by the global element) and every x
    re-uses them."""
    P = orc.Program(spec)
    n = spec.n
    N = 1 << n
    r_in = np.arange(N, dtype=np.uint64)
    r_out = r_out_for(P, n, N)
    step = max(32, N // 8)
    parts = pmap(lambda lo: P.keygen(r_in[lo:lo + step], np.ascontiguousarray(r_out[:, lo:lo + step]), seed, first_elem=lo),
                 range(0, N, step))

    def one(x):
        xv = np.full(N, x, dtype=np.uint64)
        xhat = (xv + r_in) & mask_of(n)
        for lo, (k0, k1) in zip(range(0, N, step), parts):
            sl = slice(lo, lo + step)
            out = P.run_gate(k0, k1, xhat[sl])
            check_gate_outputs(P, spec, xv[sl], r_in[sl], r_out[:, sl], out, calls)
    pmap(one, xs)
    return P


def check_pairs(orc, spec, x, r_in, seed=11, calls=True, chunk=2048):
    """Arbitrary (x, r) pairs: keygen + both calls + post for every pair, in parallel chunks."""
    P = orc.Program(spec)
    n = spec.n
    count = x.size
    r_out = r_out_for(P, n, count)

    def one(lo):
        sl = slice(lo, min(count, lo + chunk))
        ro = np.ascontiguousarray(r_out[:, sl])
        k0, k1 = P.keygen(r_in[sl], ro, seed, first_elem=lo)
        out = P.run_gate(k0, k1, (x[sl] + r_in[sl]) & mask_of(n))
        check_gate_outputs(P, spec, x[sl], r_in[sl], ro, out, calls)
    pmap(one, range(0, count, chunk))
    return P


def corner_masks(spec, extra=3, seed=0):
    """Masks that hit Protocol 3's corner cases: r = 0 and r = -alpha_i (a translated start lands on 0: the beta_0 = 0
    branch with its dummy split), r = N-1, r = N/2, plus a few seeded random ones."""
    N = 1 << spec.n
    rng = np.random.default_rng(seed)
    rs = [0, N - 1, N // 2, 1] + [(N - a) % N for a in spec.alpha] + [int(v) for v in rng.integers(0, N, extra)]
    return sorted(set(rs))


def corner_inputs(spec, extra=3, seed=0):
    """x on, just below and just above every interval boundary, the ring's ends and the sign change, plus random ones."""
    N = 1 << spec.n
    rng = np.random.default_rng(seed + 100)
    xs = [0, 1, N - 1, N // 2, N // 2 - 1]
    for a in spec.alpha:
        xs += [a, (a - 1) % N, (a + 1) % N]
    xs += [int(v) for v in rng.integers(0, N, extra)]
    return sorted(set(xs))
