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
        n_out_a, n_out_b = int(rng.integers(1, 3)), int(rng.integers(0, 4))
        for j in range(n_out_a):
            phi.append((S.PHI_A_OUT, j, int(rng.choice(A)), 0, 0))
        for j in range(n_out_b):
            phi.append((S.PHI_B_OUT, j, int(rng.choice(B)), 0, 0))
    spec = S._mk(f"rand{seed}_n{n}", n, f, cuts, coeff, nodes=nodes, bit_root=bit_root if ell else None, aux=aux if p_aux else None,
                 kappa_a=kappa_a, kappa_b=kappa_b, phi=phi, n_out_a=n_out_a, n_out_b=n_out_b,
                 mask_output=bool(rng.random() < 0.3), out_frac=f)
    spec.variant = variant if (not (variant & 4) or d <= 2) else variant & 3
    return spec
