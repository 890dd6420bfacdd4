"""Thin Python binding of libplk.so (include/plk.h): argument marshalling only.

Every function here has the name of the C entry point it calls (minus the `plk_` prefix) and does nothing but
convert numpy arrays to C pointers and raise on a negative status.  All arithmetic of the method runs in the CUDA
kernels behind the C ABI; PyTorch appears only as the owner of the device arena and of the CUDA stream.
There is NO fallback: if libplk.so is missing or does not load, importing a symbol raises.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libplk.so")

SUCCESS = 0
ERR_GENERAL, ERR_OUT_OF_MEMORY, ERR_OUT_OF_RANGE, ERR_UNINITIALIZED = -1, -2, -3, -4
ERR_UNSUPPORTED, ERR_FLOATING_POINT, ERR_CUDA, ERR_STOP_CODON = -5, -6, -7, -8
ERR_STATIC_SCRATCH_LIMIT = -9
STATIC_SCRATCH_DOUBLES, STATIC_SCALE_MAX = 8192, 2048
FP64, FP32 = 0, 1
FLAG_TENSOR_CORES, FLAG_NO_LEVEL_BATCH, FLAG_SITE_DERIVATIVES = 1, 2, 4
FLAG_LEVEL_BATCH_ONLY, FLAG_PATTERN_WALK_ONLY, FLAG_NO_TMA = 8, 16, 32
FLAG_NO_TCGEN05 = 64
FLAG_NO_PDL = 128
FLAG_CACHE_RATE_PRODUCTS, FLAG_ON_THE_FLY_MATRICES = 256, 512
NUCLEOTIDE, CODON = 0, 1


class Config(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "tip_count", "state_count", "pattern_count", "category_count", "partials_buffer_count",
        "compact_buffer_count", "partials_slot_count", "preorder_buffer_count", "preorder_slot_count",
        "matrix_buffer_count", "eigen_buffer_count", "scale_buffer_count", "precision", "flags")]


class Op(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("dest", "dest_scale", "child1", "child1_matrix", "child2", "child2_matrix")]


class PreOp(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("dest_pre", "parent_pre", "matrix", "sibling_post", "sibling_matrix",
                                         "node_post")]


OP_DTYPE = np.dtype([(n, np.int32) for n, _ in Op._fields_])
PRE_OP_DTYPE = np.dtype([(n, np.int32) for n, _ in PreOp._fields_])

_P = C.c_void_p
_I = C.c_int
_SIGNATURES = {
    "plk_arena_bytes": (C.c_size_t, [_P]),
    "plk_create": (_I, [_P, _P, C.c_size_t, _P, _P]),
    "plk_destroy": (_I, [_P]),
    "plk_error_string": (C.c_char_p, [_I]),
    "plk_set_tip_states": (_I, [_P, _I, _P]),
    "plk_set_tip_states_u8": (_I, [_P, _I, _P]),
    "plk_set_all_tip_states_u8": (_I, [_P, _P, _I]),
    "plk_set_tip_partials": (_I, [_P, _I, _P]),
    "plk_set_partials": (_I, [_P, _I, _P]),
    "plk_set_pattern_weights": (_I, [_P, _P]),
    "plk_set_state_frequencies": (_I, [_P, _P]),
    "plk_set_category_rates": (_I, [_P, _P]),
    "plk_set_category_weights": (_I, [_P, _P]),
    "plk_set_eigen_decomposition": (_I, [_P, _I, _P, _P, _P]),
    "plk_set_rate_matrix": (_I, [_P, _I, _P]),
    "plk_set_transition_matrix": (_I, [_P, _I, _P]),
    "plk_update_transition_matrices": (_I, [_P, _I, _P, _P, _I]),
    "plk_update_transition_matrices_device": (_I, [_P, _I, _P, _P, _I]),
    "plk_update_partials": (_I, [_P, _P, _I]),
    "plk_update_partials_on_the_fly": (_I, [_P, _I, _P, _I, _P]),
    "plk_cache_rate_products": (_I, [_P, _I, _P, _I]),
    "plk_root_log_likelihoods": (_I, [_P, _I, _P, _I, _P, _P]),
    "plk_root_log_likelihoods_device": (_I, [_P, _I, _P, _I, _P, _P]),
    "plk_root_log_likelihoods_static_device": (_I, [_P, _I, _P, _I, _P, _P]),
    "plk_update_pre_partials": (_I, [_P, _I, _P, _I]),
    "plk_branch_derivatives": (_I, [_P, _I, _P, _P, _I, _P, _P]),
    "plk_pre_order_gradient": (_I, [_P, _I, _I, _P, _I, _P, _P]),
    "plk_pre_order_gradient_device": (_I, [_P, _I, _I, _P, _I, _P, _P]),
    "plk_evaluate_device": (_I, [_P, _I, _P, _P, _I, _P, _I, _I, _P, _I, _I, _P, _I, _P]),
    "plk_evaluate": (_I, [_P, _I, _P, _P, _I, _P, _I, _I, _P, _I, _I, _P, _I, _P, _P]),
    "plk_rate_matrix_gradient": (_I, [_P, _P, _P, _P, _I, _P]),
    "plk_chain_rule_rate_matrix": (_I, [_P, _P, _I, _I, _P]),
    "plk_get_partials": (_I, [_P, _I, _I, _P]),
    "plk_get_scale_factors": (_I, [_P, _I, _P]),
    "plk_get_transition_matrix": (_I, [_P, _I, _P]),
    "plk_get_rate_matrix": (_I, [_P, _I, _P]),
    "plk_synchronize": (_I, [_P]),
    "plk_kernel_launch_count": (C.c_int64, [_P]),
    "plk_schedule_levels": (_I, [_P, _I, _P]),
    "plk_schedule_pre_levels": (_I, [_P, _I, _P, _P]),
    "plk_encode_and_compress": (_I, [_I, _I, C.c_int64, _P, _P, _P, _P, _P]),
}
EXPORTED = tuple(_SIGNATURES)

_lib = None


def lib():
    """The loaded libplk.so (raises OSError if it was not built: run `python -m paper_2606_27607_b200.build`)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise OSError(f"{LIB_PATH} not found: build it with `python -m paper_2606_27607_b200.build` "
                          "(there is no CPU or PyTorch fallback)")
        handle = C.CDLL(LIB_PATH)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(handle, name)  # AttributeError if a declared symbol is not exported
            fn.restype = res
            fn.argtypes = args
        _lib = handle
    return _lib


class PlkError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {error_string(status)} ({status})")


def error_string(status: int) -> str:
    return lib().plk_error_string(int(status)).decode()


def _check(status: int, where: str, allow: Sequence[int] = ()):
    if status != SUCCESS and status not in allow:
        raise PlkError(status, where)
    return status


def _f64(a, n: Optional[int] = None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if n is not None and a.size != n:
        raise ValueError(f"expected {n} values, got {a.size}")
    return a


def _i32(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def arena_bytes(cfg: Config) -> int:
    return int(lib().plk_arena_bytes(C.byref(cfg)))


def schedule_levels(ops: np.ndarray):
    """plk_schedule_levels: (n_levels, level[count]) of a post-order op list (host only)."""
    ops = np.ascontiguousarray(ops, dtype=OP_DTYPE)
    level = np.zeros(len(ops), dtype=np.int32)
    n = lib().plk_schedule_levels(_ptr(ops), len(ops), _ptr(level))
    _check(min(n, 0), "plk_schedule_levels")
    return n, level


def schedule_pre_levels(ops: np.ndarray):
    ops = np.ascontiguousarray(ops, dtype=PRE_OP_DTYPE)
    level = np.zeros(len(ops), dtype=np.int32)
    partner = np.zeros(len(ops), dtype=np.int32)
    n = lib().plk_schedule_pre_levels(_ptr(ops), len(ops), _ptr(level), _ptr(partner))
    _check(min(n, 0), "plk_schedule_pre_levels")
    return n, level, partner


def chain_rule_rate_matrix(G, dQ):
    """plk_chain_rule_rate_matrix: out[k] = sum_ab G[a][b] dQ[k][a][b] (host only)."""
    G = _f64(G)
    S = int(round(np.sqrt(G.size)))
    dQ = _f64(dQ)
    K = dQ.size // (S * S)
    out = np.zeros(K)
    _check(lib().plk_chain_rule_rate_matrix(_ptr(G), _ptr(dQ), S, K, _ptr(out)), "plk_chain_rule_rate_matrix")
    return out


def encode_and_compress(state_kind: int, seqs: Sequence[bytes]):
    """plk_encode_and_compress: (states uint8 [taxa][n_patterns], weights [n_patterns], site_to_pattern [cols])."""
    taxa = len(seqs)
    sites = len(seqs[0]) if taxa else 0
    if any(len(s) != sites for s in seqs):
        raise ValueError("sequences differ in length")
    cols = sites // 3 if state_kind == CODON else sites
    arr = (C.c_char_p * taxa)(*[bytes(s) for s in seqs])
    states = np.zeros((taxa, max(cols, 1)), dtype=np.uint8)
    weights = np.zeros(max(cols, 1), dtype=np.float64)
    s2p = np.zeros(max(cols, 1), dtype=np.int64)
    n = C.c_int64(0)
    rc = lib().plk_encode_and_compress(state_kind, taxa, sites, C.cast(arr, C.c_void_p), _ptr(states), _ptr(weights),
                                       _ptr(s2p), C.byref(n))
    _check(rc, "plk_encode_and_compress")
    k = int(n.value)
    return np.ascontiguousarray(states[:, :k]), weights[:k].copy(), s2p[:cols].copy()


class Instance:
    """One plk_instance living in a torch-owned device arena on a torch-owned stream."""

    def __init__(self, tip_count, state_count, pattern_count, category_count, *, partials_buffer_count=None,
                 compact_buffer_count=None, partials_slot_count=0, preorder_buffer_count=None,
                 preorder_slot_count=0, matrix_buffer_count=None, eigen_buffer_count=1, scale_buffer_count=None,
                 precision=FP64, flags=0, device="cuda:0", stream=None):
        import torch  # device memory and stream only

        n_nodes = 2 * tip_count - 1
        self.cfg = Config(
            tip_count, state_count, pattern_count, category_count,
            n_nodes if partials_buffer_count is None else partials_buffer_count,
            tip_count if compact_buffer_count is None else compact_buffer_count,
            partials_slot_count,
            n_nodes if preorder_buffer_count is None else preorder_buffer_count,
            preorder_slot_count,
            n_nodes if matrix_buffer_count is None else matrix_buffer_count,
            eigen_buffer_count,
            n_nodes if scale_buffer_count is None else scale_buffer_count,
            precision, flags)
        self._h = C.c_void_p(None)
        need = arena_bytes(self.cfg)
        if need == 0:
            # let plk_create say why (it distinguishes _UNSUPPORTED from _OUT_OF_RANGE)
            dummy = C.c_void_p(1024)
            _check(lib().plk_create(C.byref(self.cfg), dummy, 0, None, C.byref(self._h)), "plk_create")
            raise PlkError(ERR_OUT_OF_RANGE, "plk_arena_bytes")
        if not torch.cuda.is_available():
            raise PlkError(ERR_CUDA, "plk_create (no CUDA device; there is no CPU path)")
        self.device = torch.device(device)
        self.torch = torch
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            self.arena = torch.empty(need + 1024, dtype=torch.uint8, device=self.device)
            base = (self.arena.data_ptr() + 1023) // 1024 * 1024
            _check(lib().plk_create(C.byref(self.cfg), C.c_void_p(base), need, C.c_void_p(self.stream.cuda_stream),
                                    C.byref(self._h)), "plk_create")
        self.P, self.S, self.Cc, self.N = pattern_count, state_count, category_count, tip_count

    # -- life cycle
    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().plk_destroy(self._h)
            self._h = C.c_void_p(None)
            self.arena = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def _call(self, name, *args, allow=()):
        with self.torch.cuda.device(self.device):
            return _check(getattr(lib(), name)(self._h, *args), name, allow)

    # -- setters
    def set_tip_states(self, tip, states):
        s = _i32(states)
        if s.size != self.P:
            raise ValueError("states must have pattern_count entries")
        self._call("plk_set_tip_states", tip, _ptr(s))

    def set_tip_states_u8(self, tip, states):
        """One byte per pattern (values >= S: missing); enqueued without synchronising: `states` (a contiguous uint8
        array, ideally pinned) must stay unchanged until the next call that returns values to the host."""
        s = np.ascontiguousarray(states, dtype=np.uint8)
        if s.size != self.P:
            raise ValueError("states must have pattern_count entries")
        self._call("plk_set_tip_states_u8", tip, _ptr(s))

    def set_all_tip_states_u8(self, states):
        """plk_set_all_tip_states_u8: `states` a contiguous uint8 array [n_tips][P] (pinned memory stays valid until the
        next synchronising call); one pitched copy for tips in consecutive compact slots."""
        if states.dtype != np.uint8 or not states.flags["C_CONTIGUOUS"] or states.ndim != 2 or states.shape[1] != self.P:
            raise ValueError("states must be a C-contiguous uint8 array [n_tips][pattern_count]")
        self._call("plk_set_all_tip_states_u8", _ptr(states), states.shape[0])

    def set_tip_partials(self, tip, partials):
        self._call("plk_set_tip_partials", tip, _ptr(_f64(partials, self.P * self.S)))

    def set_partials(self, buffer, partials):
        self._call("plk_set_partials", buffer, _ptr(_f64(partials, self.Cc * self.P * self.S)))

    def set_pattern_weights(self, w):
        self._call("plk_set_pattern_weights", _ptr(_f64(w, self.P)))

    def set_state_frequencies(self, pi):
        self._call("plk_set_state_frequencies", _ptr(_f64(pi, self.S)))

    def set_category_rates(self, r):
        self._call("plk_set_category_rates", _ptr(_f64(r, self.Cc)))

    def set_category_weights(self, w):
        self._call("plk_set_category_weights", _ptr(_f64(w, self.Cc)))

    def set_eigen_decomposition(self, eigen, U, Uinv, lam):
        S = self.S
        self._call("plk_set_eigen_decomposition", eigen, _ptr(_f64(U, S * S)), _ptr(_f64(Uinv, S * S)),
                   _ptr(_f64(lam, S)))

    def set_rate_matrix(self, eigen, Q):
        self._call("plk_set_rate_matrix", eigen, _ptr(_f64(Q, self.S * self.S)))

    def set_transition_matrix(self, matrix, m):
        self._call("plk_set_transition_matrix", matrix, _ptr(_f64(m, self.Cc * self.S * self.S)))

    # -- hot path
    def update_transition_matrices(self, eigen, matrix_idx, branch_lengths):
        idx = _i32(matrix_idx)
        t = _f64(branch_lengths, idx.size)
        self._call("plk_update_transition_matrices", eigen, _ptr(idx), _ptr(t), idx.size)

    def update_transition_matrices_device(self, eigen, matrix_idx, d_branch_lengths):
        """d_branch_lengths: torch fp64 CUDA tensor [count]."""
        idx = _i32(matrix_idx)
        self._call("plk_update_transition_matrices_device", eigen, _ptr(idx), C.c_void_p(d_branch_lengths.data_ptr()),
                   idx.size)

    def update_partials(self, ops):
        ops = np.ascontiguousarray(ops, dtype=OP_DTYPE)
        self._call("plk_update_partials", _ptr(ops), len(ops))

    def root_log_likelihoods(self, root_buffer, scale_idx, want_site=True, allow_nonfinite=False):
        sc = _i32(scale_idx)
        out_sum = np.zeros(1)
        out_site = np.zeros(self.P) if want_site else None
        self._call("plk_root_log_likelihoods", root_buffer, _ptr(sc), sc.size, _ptr(out_sum), _ptr(out_site),
                   allow=(ERR_FLOATING_POINT,) if allow_nonfinite else ())
        return float(out_sum[0]), out_site

    def root_log_likelihoods_device(self, root_buffer, scale_idx, d_out_sum, d_out_site=None):
        sc = _i32(scale_idx)
        self._call("plk_root_log_likelihoods_device", root_buffer, _ptr(sc), sc.size, C.c_void_p(d_out_sum.data_ptr()),
                   None if d_out_site is None else C.c_void_p(d_out_site.data_ptr()))

    def root_log_likelihoods_static_device(self, root_buffer, scale_idx, d_out_sum, d_out_site=None):
        """plk_root_log_likelihoods_static_device: the same reduction with its scratch in the library's static device
        array (no allocation; limits STATIC_SCRATCH_DOUBLES / STATIC_SCALE_MAX)."""
        sc = _i32(scale_idx)
        self._call("plk_root_log_likelihoods_static_device", root_buffer, _ptr(sc), sc.size,
                   C.c_void_p(d_out_sum.data_ptr()), None if d_out_site is None else C.c_void_p(d_out_site.data_ptr()))

    def update_pre_partials(self, root_pre_buffer, ops):
        ops = np.ascontiguousarray(ops, dtype=PRE_OP_DTYPE)
        self._call("plk_update_pre_partials", root_pre_buffer, _ptr(ops), len(ops))

    def branch_derivatives(self, eigen, post_idx, pre_idx, want_site=False):
        a, b = _i32(post_idx), _i32(pre_idx)
        grad = np.zeros(a.size)
        site = np.zeros((a.size, self.P)) if want_site else None
        self._call("plk_branch_derivatives", eigen, _ptr(a), _ptr(b), a.size, _ptr(grad), _ptr(site))
        return grad, site

    def pre_order_gradient(self, eigen, root_pre_buffer, ops, want_site=False):
        ops = np.ascontiguousarray(ops, dtype=PRE_OP_DTYPE)
        grad = np.zeros(len(ops))
        site = np.zeros((len(ops), self.P)) if want_site else None
        self._call("plk_pre_order_gradient", eigen, root_pre_buffer, _ptr(ops), len(ops), _ptr(grad), _ptr(site))
        return grad, site

    def pre_order_gradient_device(self, eigen, root_pre_buffer, ops, d_out_gradient, d_out_site=None):
        ops = np.ascontiguousarray(ops, dtype=PRE_OP_DTYPE)
        self._call("plk_pre_order_gradient_device", eigen, root_pre_buffer, _ptr(ops), len(ops),
                   C.c_void_p(d_out_gradient.data_ptr()),
                   None if d_out_site is None else C.c_void_p(d_out_site.data_ptr()))

    def update_partials_on_the_fly(self, eigen, ops, branch_lengths):
        """plk_update_partials_on_the_fly: branch_lengths [count][2] = lengths of the branches above child1 / child2."""
        ops = np.ascontiguousarray(ops, dtype=OP_DTYPE)
        t = _f64(branch_lengths, 2 * len(ops))
        self._call("plk_update_partials_on_the_fly", eigen, _ptr(ops), len(ops), _ptr(t))

    def cache_rate_products(self, eigen, post_idx):
        a = _i32(post_idx)
        self._call("plk_cache_rate_products", eigen, _ptr(a), a.size)

    def evaluate_device(self, eigen, matrix_idx, d_branch_lengths, ops, root_buffer, scale_idx, root_pre_buffer, pre_ops,
                        d_out):
        """plk_evaluate_device: steps 1-6 in one call (cached CUDA graph); d_out = [logL, gradient] on the device."""
        m, sc = _i32(matrix_idx), _i32(scale_idx)
        ops = np.ascontiguousarray(ops, dtype=OP_DTYPE)
        pre = np.ascontiguousarray(pre_ops, dtype=PRE_OP_DTYPE)
        self._call("plk_evaluate_device", eigen, _ptr(m), C.c_void_p(d_branch_lengths.data_ptr()), m.size, _ptr(ops),
                   len(ops), root_buffer, _ptr(sc), sc.size, root_pre_buffer, _ptr(pre), len(pre),
                   C.c_void_p(d_out.data_ptr()))

    def evaluate(self, eigen, matrix_idx, branch_lengths, ops, root_buffer, scale_idx, root_pre_buffer, pre_ops,
                 allow_nonfinite=False):
        """plk_evaluate: the same with host branch lengths in, (logL, gradient[len(pre_ops)]) out."""
        m, sc = _i32(matrix_idx), _i32(scale_idx)
        t = _f64(branch_lengths, m.size)
        ops = np.ascontiguousarray(ops, dtype=OP_DTYPE)
        pre = np.ascontiguousarray(pre_ops, dtype=PRE_OP_DTYPE)
        logl = np.zeros(1)
        grad = np.zeros(len(pre))
        self._call("plk_evaluate", eigen, _ptr(m), _ptr(t), m.size, _ptr(ops), len(ops), root_buffer, _ptr(sc), sc.size,
                   root_pre_buffer, _ptr(pre), len(pre), _ptr(logl), _ptr(grad),
                   allow=(ERR_FLOATING_POINT,) if allow_nonfinite else ())
        return float(logl[0]), grad

    def rate_matrix_gradient(self, post_idx, pre_idx, branch_lengths):
        a, b = _i32(post_idx), _i32(pre_idx)
        t = _f64(branch_lengths, a.size)
        out = np.zeros((self.S, self.S))
        self._call("plk_rate_matrix_gradient", _ptr(a), _ptr(b), _ptr(t), a.size, _ptr(out))
        return out

    # -- read-back
    def get_partials(self, buffer, pre=False):
        """pre: False / 0 post-order, True / 1 pre-order, 2 the cached rate product Q p_k of a post-order buffer."""
        out = np.zeros((self.Cc, self.P, self.S))
        self._call("plk_get_partials", buffer, int(pre), _ptr(out))
        return out

    def get_scale_factors(self, scale):
        out = np.zeros(self.P)
        self._call("plk_get_scale_factors", scale, _ptr(out))
        return out

    def get_transition_matrix(self, matrix):
        out = np.zeros((self.Cc, self.S, self.S))
        self._call("plk_get_transition_matrix", matrix, _ptr(out))
        return out

    def get_rate_matrix(self, eigen):
        out = np.zeros((self.S, self.S))
        self._call("plk_get_rate_matrix", eigen, _ptr(out))
        return out

    def synchronize(self):
        self._call("plk_synchronize")

    def kernel_launch_count(self) -> int:
        return int(lib().plk_kernel_launch_count(self._h))
