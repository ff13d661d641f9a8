"""fusefss-b200: thin ctypes binding over libfusefss.so (C ABI in include/fusefss.h).

Argument marshalling only -- every step of the hot path (keygen, eval_cmp, eval_lut, post) runs inside the
library's sm_100a kernels.  PyTorch supplies device memory and streams.  There is NO CPU fallback: if the
shared library is missing the import fails, and every compute call needs a CUDA device.
Functions carry the same names as the C ABI (`fusefss_compile`, `fusefss_keygen`, ...); `Program` is a
convenience wrapper that allocates the output tensors.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfusefss.so")

# every symbol include/fusefss.h declares (tests check the library exports all of them)
SYMBOLS = (
    "fusefss_compile", "fusefss_destroy", "fusefss_prepare", "fusefss_shape", "fusefss_atom", "fusefss_key_bytes", "fusefss_keygen", "fusefss_keygen_parts",
    "fusefss_eval_cmp", "fusefss_eval_lut", "fusefss_eval_fused", "fusefss_eval_fused_both", "fusefss_post", "fusefss_post_rounds", "fusefss_post_msg_bytes",
    "fusefss_online_bits", "fusefss_post_fused", "fusefss_post_fused_noalloc", "fusefss_cost", "fusefss_gate_workspace_bytes", "fusefss_gate_host",
    "fusefss_share_open", "fusefss_open_output", "fusefss_sub_bcast", "fusefss_row_sum", "fusefss_mul_triple_bytes", "fusefss_mul_keygen", "fusefss_mul_fused",
    "fusefss_strerror", "fusefss_last_cuda_error", "fusefss_debug_set", "fusefss_launch_count", "fusefss_aes_probe", "fusefss_aes_chain_probe", "fusefss_aes_kat", "fusefss_pipe_probe", "fusefss_bitslice_kat", "fusefss_bitslice_probe",
)


class BitNode(C.Structure):
    _fields_ = [("kind", C.c_uint8), ("k", C.c_uint8), ("lhs", C.c_uint16), ("rhs", C.c_uint16),
                ("value_is_2k", C.c_uint8), ("pad", C.c_uint8), ("value", C.c_uint64)]


class Kappa(C.Structure):
    _fields_ = [("kind", C.c_uint8), ("arg", C.c_uint8)]


class PhiOp(C.Structure):
    _fields_ = [("op", C.c_uint8), ("dst", C.c_uint8), ("a", C.c_uint8), ("b", C.c_uint8), ("pad", C.c_uint32),
                ("imm", C.c_uint64)]


class Spec(C.Structure):
    _fields_ = [(k, C.c_uint32) for k in ("n", "frac_bits", "m", "r", "d", "p_aux", "ell", "n_nodes", "n_kappa_a",
                                          "n_kappa_b", "phi_len", "n_out_a", "n_out_b", "mask_output", "variant")] + \
               [(k, C.c_void_p) for k in ("alpha", "coeff", "aux", "nodes", "bit_root", "kappa_a", "kappa_b", "phi")]


class Cost(C.Structure):
    _fields_ = [(k, C.c_uint64) for k in ("eval_cmp_aes", "eval_cmp_lookups", "eval_lut_aes", "eval_lut_lookups", "gen_cmp_aes",
                                          "gen_cmp_lookups", "gen_lut_aes", "gen_lut_lookups", "eval_cmp_key_bytes",
                                          "eval_lut_key_bytes")]


class Shape(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("T", "M", "p", "M_A", "M_B", "G_mix", "rounds", "n_out_a", "n_out_b",
                                         "has_lut", "n_kb")] + [("k", C.c_int32 * 64)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                          "(nvcc, sm_100a).  There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, u64, sz, i32 = C.c_void_p, C.c_uint64, C.c_size_t, C.c_int
    sig = {
        "fusefss_compile": (i32, [C.POINTER(Spec), C.POINTER(vp)]),
        "fusefss_destroy": (None, [vp]),
        "fusefss_prepare": (i32, [vp]),
        "fusefss_shape": (i32, [vp, C.POINTER(Shape)]),
        "fusefss_atom": (i32, [vp, i32, C.POINTER(u64)]),
        "fusefss_key_bytes": (sz, [vp, sz]),
        "fusefss_keygen": (i32, [vp, vp, vp, u64, u64, sz, vp, vp, vp]),
        "fusefss_keygen_parts": (i32, [vp, vp, vp, u64, u64, sz, vp, vp, i32, vp]),
        "fusefss_eval_cmp": (i32, [i32, vp, vp, vp, sz, vp, vp]),
        "fusefss_eval_lut": (i32, [i32, vp, vp, vp, sz, vp, vp]),
        "fusefss_eval_fused": (i32, [i32, vp, vp, vp, sz, vp, vp, vp]),
        "fusefss_eval_fused_both": (i32, [vp, vp, vp, vp, sz, vp, vp, vp, vp, vp]),
        "fusefss_post": (i32, [i32, vp, vp, vp, vp, vp, sz, i32, vp, vp, vp, vp, vp]),
        "fusefss_post_rounds": (i32, [vp]),
        "fusefss_post_msg_bytes": (sz, [vp, sz, i32]),
        "fusefss_online_bits": (sz, [vp]),
        "fusefss_post_fused": (i32, [vp, vp, vp, vp, vp, vp, vp, vp, sz, vp, vp, vp, vp, vp]),
        "fusefss_post_fused_noalloc": (i32, [vp, vp, vp, vp, vp, vp, vp, vp, sz, vp, vp, vp, vp, vp]),
        "fusefss_cost": (i32, [vp, C.POINTER(Cost)]),
        "fusefss_gate_workspace_bytes": (sz, [vp, sz]),
        "fusefss_gate_host": (i32, [vp, vp, vp, vp, u64, sz, sz, vp, sz, vp, vp, vp, vp, vp]),
        "fusefss_share_open": (i32, [vp, vp, vp, vp, vp, sz, u64, vp, vp]),
        "fusefss_open_output": (i32, [C.c_uint32, vp, vp, sz, u64, vp, vp]),
        "fusefss_sub_bcast": (i32, [C.c_uint32, vp, vp, sz, sz, vp, vp]),
        "fusefss_row_sum": (i32, [C.c_uint32, vp, sz, sz, vp, vp]),
        "fusefss_mul_triple_bytes": (sz, [sz]),
        "fusefss_mul_keygen": (i32, [C.c_uint32, u64, u64, sz, vp, vp, vp]),
        "fusefss_mul_fused": (i32, [C.c_uint32, vp, vp, vp, vp, vp, vp, sz, sz, vp, vp, vp]),
        "fusefss_strerror": (C.c_char_p, [i32]),
        "fusefss_last_cuda_error": (C.c_char_p, []),
        "fusefss_debug_set": (i32, [C.c_char_p, C.c_long]),
        "fusefss_launch_count": (u64, []),
        "fusefss_aes_probe": (i32, [sz, i32, vp, vp]),
        "fusefss_aes_chain_probe": (i32, [i32, i32, vp, vp]),
        "fusefss_aes_kat": (i32, [C.c_char_p, C.c_char_p, vp, vp]),
        "fusefss_pipe_probe": (i32, [i32, i32, vp, vp]),
        "fusefss_bitslice_kat": (i32, [C.c_char_p, vp, vp, vp]),
        "fusefss_bitslice_probe": (i32, [C.c_char_p, sz, i32, vp, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    return L


lib = _load()


class FuseFSSError(RuntimeError):
    pass


def _check(rc: int):
    if rc != 0:
        msg = lib.fusefss_strerror(rc).decode()
        if rc == -6:
            msg += ": " + lib.fusefss_last_cuda_error().decode()
        raise FuseFSSError(f"libfusefss error {rc}: {msg}")


def _ptr(t):
    """device (or pinned host) pointer of a torch tensor / numpy array, or NULL"""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p) if a is not None and a.size else None


class _SpecHolder:
    """workloads.specs.OpSpec -> fusefss_spec (keeps the host arrays alive)"""

    def __init__(self, s):
        u = lambda a: np.ascontiguousarray(np.asarray(a, dtype=np.uint64)).reshape(-1)
        self.alpha, self.coeff, self.aux = u(s.alpha), u(s.coeff), u(s.aux)
        self.nodes = (BitNode * max(1, len(s.nodes)))(*[BitNode(kind, k, lhs, rhs, is2k, 0, value)
                                                        for (kind, k, lhs, rhs, is2k, value) in s.nodes])
        self.bit_root = np.ascontiguousarray(np.asarray(s.bit_root, dtype=np.uint16)).reshape(-1)
        self.ka = (Kappa * max(1, len(s.kappa_a)))(*[Kappa(*k) for k in s.kappa_a])
        self.kb = (Kappa * max(1, len(s.kappa_b)))(*[Kappa(*k) for k in s.kappa_b])
        self.phi = (PhiOp * max(1, len(s.phi)))(*[PhiOp(op, dst, a, b, 0, imm & 0xFFFFFFFFFFFFFFFF)
                                                  for (op, dst, a, b, imm) in s.phi])
        self.c = Spec(s.n, s.f, s.m, s.r, s.d, s.p_aux, s.ell, len(s.nodes), len(s.kappa_a), len(s.kappa_b),
                      len(s.phi), s.n_out_a, s.n_out_b, int(s.mask_output), int(getattr(s, "variant", 0)),
                      _np_ptr(self.alpha), _np_ptr(self.coeff), _np_ptr(self.aux), C.cast(self.nodes, C.c_void_p),
                      _np_ptr(self.bit_root), C.cast(self.ka, C.c_void_p), C.cast(self.kb, C.c_void_p),
                      C.cast(self.phi, C.c_void_p))


SHAPE_KEYS = ("T", "M", "p", "M_A", "M_B", "G_mix", "rounds", "n_out_a", "n_out_b", "has_lut", "n_kb")


class Program:
    """A compiled gate type (fusefss_compile).  Tensors are torch uint64-as-int64 CUDA tensors; the methods
    allocate outputs and forward raw pointers + the current stream to the C ABI."""

    def __init__(self, spec):
        self.spec = spec
        self._holder = _SpecHolder(spec)
        h = C.c_void_p()
        _check(lib.fusefss_compile(C.byref(self._holder.c), C.byref(h)))
        self._h = h
        sh = Shape()
        _check(lib.fusefss_shape(self._h, C.byref(sh)))
        self.shape = {k: int(getattr(sh, k)) for k in SHAPE_KEYS}
        self.shape["k"] = [int(sh.k[t]) for t in range(self.shape["T"])]

    def __del__(self):
        if getattr(self, "_h", None) and lib is not None:       # `lib` is gone at interpreter shutdown
            lib.fusefss_destroy(self._h)
            self._h = None

    # ---- host-side queries -------------------------------------------------------------------
    def atom(self, t):
        out = (C.c_uint64 * 4)()
        _check(lib.fusefss_atom(self._h, t, out))
        return dict(k=int(out[0]), c=int(out[1]), is_theta=int(out[2]), beta=int(out[3]))

    def key_bytes(self, count):
        return lib.fusefss_key_bytes(self._h, count)

    def post_rounds(self):
        return lib.fusefss_post_rounds(self._h)

    def post_msg_bytes(self, count, rnd):
        return lib.fusefss_post_msg_bytes(self._h, count, rnd)

    def msg_total(self, count):
        return sum(self.post_msg_bytes(count, q) for q in range(self.post_rounds()))

    def online_bits(self):
        return lib.fusefss_online_bits(self._h)

    def cost(self):
        c = Cost()
        _check(lib.fusefss_cost(self._h, C.byref(c)))
        return {k: int(getattr(c, k)) for k, _ in Cost._fields_}

    def prepare(self):
        """fusefss_prepare: upload the program's tables to the current device now instead of on first use"""
        _check(lib.fusefss_prepare(self._h))
        return self

    def workspace_bytes(self, chunk):
        return lib.fusefss_gate_workspace_bytes(self._h, chunk)

    # ---- device calls ------------------------------------------------------------------------
    @staticmethod
    def _empty(shape, dtype=None):
        import torch
        return torch.empty(shape, dtype=dtype or torch.int64, device="cuda")

    def alloc_keys(self, count):
        import torch
        kb = self.key_bytes(count)
        return (torch.empty(kb, dtype=torch.uint8, device="cuda"), torch.empty(kb, dtype=torch.uint8, device="cuda"))

    def keygen(self, r_in, r_out, seed, first_elem=0, keys=None, parts=7):
        count = r_in.numel()
        k0, k1 = keys if keys is not None else self.alloc_keys(count)
        if parts == 7:
            _check(lib.fusefss_keygen(self._h, _ptr(r_in), _ptr(r_out), seed, first_elem, count, _ptr(k0), _ptr(k1), _stream()))
        else:
            _check(lib.fusefss_keygen_parts(self._h, _ptr(r_in), _ptr(r_out), seed, first_elem, count, _ptr(k0), _ptr(k1),
                                            parts, _stream()))
        return k0, k1

    def eval_cmp(self, party, key, xhat, out=None):
        count = xhat.numel()
        out = self._empty(count) if out is None else out
        _check(lib.fusefss_eval_cmp(party, self._h, _ptr(key), _ptr(xhat), count, _ptr(out), _stream()))
        return out

    def eval_lut(self, party, key, xhat, out=None):
        count = xhat.numel()
        out = self._empty((self.shape["p"], count)) if out is None else out
        _check(lib.fusefss_eval_lut(party, self._h, _ptr(key), _ptr(xhat), count, _ptr(out), _stream()))
        return out

    def eval_fused(self, party, key, xhat, bits=None, coeff=None):
        count = xhat.numel()
        bits = self._empty(count) if bits is None and self.shape["T"] else bits
        coeff = self._empty((self.shape["p"], count)) if coeff is None and self.shape["has_lut"] else coeff
        _check(lib.fusefss_eval_fused(party, self._h, _ptr(key), _ptr(xhat), count, _ptr(bits), _ptr(coeff), _stream()))
        return bits, coeff

    def eval_fused_both(self, key0, key1, xhat, bits=None, coeff=None):
        count = xhat.numel()
        bits = [self._empty(count), self._empty(count)] if bits is None and self.shape["T"] else (bits or [None, None])
        coeff = ([self._empty((self.shape["p"], count)) for _ in (0, 1)] if coeff is None and self.shape["has_lut"]
                 else (coeff or [None, None]))
        _check(lib.fusefss_eval_fused_both(self._h, _ptr(key0), _ptr(key1), _ptr(xhat), count, _ptr(bits[0]), _ptr(bits[1]),
                                           _ptr(coeff[0]), _ptr(coeff[1]), _stream()))
        return bits, coeff

    def post(self, party, key, xhat, bits, coeff, rnd, msg_in, msg_out, y=None, z=None):
        count = xhat.numel()
        if rnd == self.post_rounds():
            y = self._empty((max(1, self.shape["n_out_a"]), count)) if y is None else y
            z = self._empty(count) if z is None else z
        _check(lib.fusefss_post(party, self._h, _ptr(key), _ptr(xhat), _ptr(bits), _ptr(coeff), count, rnd,
                                _ptr(msg_in), _ptr(msg_out), _ptr(y), _ptr(z), _stream()))
        return y, z

    def post_fused(self, key0, key1, xhat, bits0, bits1, coeff0, coeff1, outs=None):
        count = xhat.numel()
        na = max(1, self.shape["n_out_a"])
        y0, y1, z0, z1 = outs if outs is not None else (self._empty((na, count)), self._empty((na, count)),
                                                        self._empty(count), self._empty(count))
        _check(lib.fusefss_post_fused(self._h, _ptr(key0), _ptr(key1), _ptr(xhat), _ptr(bits0), _ptr(bits1),
                                      _ptr(coeff0), _ptr(coeff1), count, _ptr(y0), _ptr(y1), _ptr(z0), _ptr(z1), _stream()))
        return y0, y1, z0, z1

    def post_fused_noalloc(self, key0, key1, xhat, bits0, bits1, coeff0, coeff1, outs):
        """fusefss_post_fused_noalloc: post_fused for hosts that must not allocate device memory (see include/fusefss.h).
        To keep that promise on this side of the ABI too, the binding allocates nothing: `outs` = (y0, y1, z0, z1) are the
        caller's tensors.  Calls share one table per device -- keep them on one stream."""
        y0, y1, z0, z1 = outs
        _check(lib.fusefss_post_fused_noalloc(self._h, _ptr(key0), _ptr(key1), _ptr(xhat), _ptr(bits0), _ptr(bits1),
                                              _ptr(coeff0), _ptr(coeff1), xhat.numel(), _ptr(y0), _ptr(y1), _ptr(z0), _ptr(z1),
                                              _stream()))
        return y0, y1, z0, z1

    def run_gate(self, key0, key1, xhat):
        """Both parties, the two FSS calls and the per-round post API (message buffers swapped on device)."""
        import torch
        count = xhat.numel()
        keys = (key0, key1)
        T, lut = self.shape["T"], self.shape["has_lut"]
        bits = [self.eval_cmp(b, keys[b], xhat) if T else None for b in (0, 1)]
        coeff = [self.eval_lut(b, keys[b], xhat) if lut else None for b in (0, 1)]
        R = self.post_rounds()
        tot = max(256, self.msg_total(count))
        msg = [torch.zeros(tot, dtype=torch.uint8, device="cuda") for _ in (0, 1)]
        for q in range(R):
            for b in (0, 1):
                self.post(b, keys[b], xhat, bits[b], coeff[b], q, msg[1 - b], msg[b])
        outs = [self.post(b, keys[b], xhat, bits[b], coeff[b], R, msg[1 - b], msg[b]) for b in (0, 1)]
        return dict(bits=bits, coeff=coeff, msg=msg, y=[outs[0][0], outs[1][0]], z=[outs[0][1], outs[1][1]])

    def gate_host(self, r_in, r_out, xhat, seed, chunk, workspace):
        """End-to-end call with HOST (numpy / pinned) buffers: H2D, keygen, eval x2 parties, post, D2H."""
        count = int(xhat.size)
        na = max(1, self.shape["n_out_a"])
        y0 = np.empty((na, count), np.uint64); y1 = np.empty((na, count), np.uint64)
        z0 = np.zeros(count, np.uint64); z1 = np.zeros(count, np.uint64)
        _check(lib.fusefss_gate_host(self._h, _ptr(r_in), _ptr(r_out), _ptr(xhat), seed, count, chunk, _ptr(workspace),
                                     workspace.numel() * workspace.element_size(), _ptr(y0), _ptr(y1), _ptr(z0), _ptr(z1), _stream()))
        return y0, y1, z0, z1


def debug_set(knob: str, value: int):
    _check(lib.fusefss_debug_set(knob.encode(), int(value)))


def launch_count() -> int:
    return int(lib.fusefss_launch_count())


def aes_kat(key: bytes, block: bytes) -> bytes:
    import torch
    out = torch.zeros(16, dtype=torch.uint8, device="cuda")
    _check(lib.fusefss_aes_kat(key, block, _ptr(out), _stream()))
    return bytes(out.cpu().numpy().tobytes())


def bitslice_kat(key: bytes, blocks: bytes) -> bytes:
    """32 blocks (512 bytes) through the bitsliced core; returns the 512 ciphertext bytes"""
    import torch
    assert len(blocks) == 512
    src = torch.frombuffer(bytearray(blocks), dtype=torch.uint8).cuda()
    out = torch.zeros(512, dtype=torch.uint8, device="cuda")
    _check(lib.fusefss_bitslice_kat(key, _ptr(src), _ptr(out), _stream()))
    return bytes(out.cpu().numpy().tobytes())


def bitslice_probe(threads: int = 0, iters: int = 24):
    """GAES/s of the bitsliced core (CUDA events), for bench.py's prg_probe"""
    import torch
    sms = torch.cuda.get_device_properties(torch.cuda.current_device()).multi_processor_count
    threads = threads or sms * 512
    out = torch.empty(threads * 16, dtype=torch.uint8, device="cuda")
    key = bytes(range(16))
    _check(lib.fusefss_bitslice_probe(key, threads, 2, _ptr(out), _stream()))
    torch.cuda.synchronize()
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record()
    _check(lib.fusefss_bitslice_probe(key, threads, iters, _ptr(out), _stream()))
    b.record()
    torch.cuda.synchronize()
    return {"gaes": threads * 32 * iters / (a.elapsed_time(b) * 1e-3) / 1e9,
            "what": "fusefss_bitslice_probe: 32 blocks per thread as 128 bit-planes, composite-field S-box circuit (152 XOR + 36 AND per byte), no tables"}


def aes_chain_probe(blocks_per_trip: int, trips: int, out):
    """fusefss_aes_chain_probe: one warp, `trips` dependent trips of `blocks_per_trip` AES blocks; out = 512-byte CUDA tensor"""
    _check(lib.fusefss_aes_chain_probe(blocks_per_trip, trips, _ptr(out), _stream()))
    return out


def aes_probe(threads: int, iters: int, out=None):
    import torch
    out = torch.empty(threads * 16, dtype=torch.uint8, device="cuda") if out is None else out
    _check(lib.fusefss_aes_probe(threads, iters, _ptr(out), _stream()))
    return out
