"""ctypes binding of libcacheweaver.so — argument marshalling only; every step of the path runs in the library.

The function names are those of include/cacheweaver.h.  PyTorch is used for device memory and streams.
There is no fallback: if the library is missing or a kernel is requested without CUDA, this raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libcacheweaver.so")

CW_OK, CW_ERR_INVALID, CW_ERR_NO_SPACE, CW_ERR_BAD_HANDLE, CW_ERR_CUDA = 0, -1, -2, -3, -4
BLOCK_SIZE = 16
STATIC_WORK_INTS = 8 * 65536          # CW_STATIC_WORK_INTS (cacheweaver.h): capacity of cw_prefill_attn_static
ARMS = {"retrieval": 0, "greedy": 1, "sorted": 2, "recency": 3, "exhaustive": 4,      # CW_ARM_* (cacheweaver.h)
        "greedy_feedback": 5, "greedy_resident": 6}


class CwConfig(C.Structure):
    _fields_ = [("block_size", C.c_int32), ("num_blocks", C.c_int32), ("num_q_heads", C.c_int32),
                ("num_kv_heads", C.c_int32), ("head_dim", C.c_int32), ("max_position", C.c_int32),
                ("rope_theta", C.c_double), ("recency_window", C.c_int32), ("eager_register", C.c_int32),
                ("hash_salt", C.c_uint64), ("k_pool", C.c_void_p), ("v_pool", C.c_void_p),
                ("rope_table", C.c_void_p), ("device", C.c_int32), ("index_key_bits", C.c_int32)]


class CwStats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("requests", "hit_blocks", "miss_blocks", "evictions", "trie_nodes",
                                          "order_probes", "free_blocks", "seq", "predicted_prefix_docs",
                                          "actual_prefix_docs", "over_predicted_docs", "stale_marks", "prompt_tokens",
                                          "suffix_tokens", "attn_flops", "append_bytes")]


class CwError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"cacheweaver error {code}: {msg}")
        self.code = code


class NoSpace(CwError):
    pass


_lib = None


def load_library(build_if_missing: bool = True):
    """dlopen libcacheweaver.so.  The library is (re)built in-tree with nvcc whenever its source-hash stamp does not match
    the sources (a missing or stale binary is never used silently).  Fails loudly otherwise."""
    global _lib
    if _lib is not None:
        return _lib
    from .build import _stale, build
    if _stale():
        if not build_if_missing:
            raise OSError(f"{LIB_PATH} is missing or older than its sources; run python -m paper_2606_19667_b200.build")
        build()
    lib = C.CDLL(LIB_PATH)
    i32, i64, vp = C.c_int32, C.c_int64, C.c_void_p
    p = lambda _t: vp      # typed pointers are passed as plain addresses (numpy: a.ctypes.data): cheapest marshalling
    sig = {
        "cw_create": (C.c_int, [p(CwConfig), p(vp)]),
        "cw_destroy": (None, [vp]),
        "cw_strerror": (C.c_char_p, [C.c_int]),
        "cw_last_error": (C.c_char_p, [vp]),
        "cw_stats": (C.c_int, [vp, p(CwStats)]),
        "cw_pool_bytes": (i64, [p(CwConfig)]),
        "cw_pool_offset": (i64, [p(CwConfig), i32, i32, i32, i32]),
        "cw_q_roped_offset": (i64, [p(CwConfig), i32, i32, i32, i32]),
        "cw_order": (C.c_int, [vp, p(i64), i32, p(i64), p(i32)]),
        "cw_predict": (C.c_int, [vp, p(i64), i32, p(i32)]),
        "cw_order_arm": (C.c_int, [vp, i32, p(i64), i32, p(i32), i32, i32, p(i32), i32, p(i64), p(i32)]),
        "cw_observe": (C.c_int, [vp, p(i64), i32]),
        "cw_mark_stale": (C.c_int, [vp, p(i64), i32, i32]),
        "cw_feedback": (C.c_int, [vp, p(i64), i32, i32, i32]),
        "cw_matched_docs": (C.c_int, [vp, p(i32), i32, i32, i32, p(i32)]),
        "cw_feedback_tokens": (C.c_int, [vp, p(i64), i32, i32, p(i32), i32, i32, p(i32)]),
        "cw_hash_chain": (C.c_int, [vp, p(i32), i32, p(C.c_uint64)]),
        "cw_lookup": (C.c_int, [vp, p(i32), i32, i32, p(i64), p(i32), p(i32)]),
        "cw_release": (C.c_int, [vp, i64]),
        "cw_extend": (C.c_int, [vp, i64, p(i32), i32, p(i32), i32, p(i32)]),
        "cw_free_list": (C.c_int, [vp, p(i32), i32, p(i32)]),
        "cw_reset": (C.c_int, [vp]),
        "cw_admit_batch": (C.c_int, [vp, p(i64), i32, i32, i32, p(i32), i32, i32, p(i32), i32, p(i64), p(i32), p(i64),
                                     p(i32), i32, p(i32), p(i32), p(i32)]),
        "cw_release_batch": (C.c_int, [vp, p(i64), i32]),
        "cw_append_kv": (C.c_int, [vp, vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, vp]),
        "cw_attn_work_ints": (i64, [vp, i32, i32]),
        "cw_prefill_attn": (C.c_int, [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]),
        "cw_attn_schedule": (C.c_int, [vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]),
        "cw_attn_run": (C.c_int, [vp, vp, vp, vp, i32, i32, i32, vp, vp]),
        "cw_prefill_attn_static": (C.c_int, [vp, vp, vp, vp, vp, vp, vp, i32, i32, i32, i32, i32, vp, vp]),
        "cw_prefill_requests_ws_bytes": (i64, [vp, i32, i32, i32]),
        "cw_prefill_requests_work_offset": (i64, [vp, i32, i32]),
        "cw_prefill_requests": (C.c_int, [vp, p(i64), i32, vp, vp, vp, vp, vp, i32, i32, vp, vp]),
        "cw_gather_kv": (C.c_int, [vp, vp, i32, vp, vp, vp]),
        "cw_prefill_host_ws_bytes": (i64, [vp, i32, i32, i32]),
        "cw_prefill_host": (C.c_int, [vp, vp, vp, vp, vp, p(i32), p(i32), p(i32), i32, i32, i32, vp, vp]),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype, f.argtypes = res, args
    _lib = lib
    return lib


EXPORTS = ["cw_create", "cw_destroy", "cw_strerror", "cw_last_error", "cw_stats", "cw_pool_bytes", "cw_pool_offset", "cw_q_roped_offset",
           "cw_order", "cw_predict", "cw_order_arm", "cw_observe", "cw_mark_stale", "cw_feedback", "cw_matched_docs", "cw_feedback_tokens", "cw_hash_chain", "cw_lookup", "cw_release", "cw_extend", "cw_free_list",
           "cw_reset", "cw_admit_batch", "cw_release_batch",
           "cw_append_kv", "cw_attn_work_ints", "cw_prefill_attn", "cw_attn_schedule", "cw_attn_run", "cw_prefill_attn_static", "cw_prefill_requests_ws_bytes",
           "cw_prefill_requests_work_offset", "cw_prefill_requests", "cw_gather_kv", "cw_prefill_host_ws_bytes",
           "cw_prefill_host"]


def _i32p(a):
    return a.ctypes.data


def _i64p(a):
    return a.ctypes.data


def _np_i32(x):
    return np.ascontiguousarray(x, dtype=np.int32)


class Context:
    """One cw_ctx.  device=None -> host-only context (ordering + prefix cache, no kernels, no CUDA needed)."""

    def __init__(self, num_blocks, num_q_heads, num_kv_heads, head_dim, recency_window, rope_theta=10000.0,
                 max_position=0, eager_register=True, hash_salt=0, device=None, index_key_bits=0):
        self.lib = load_library()
        self.device = device
        self.Hq, self.Hkv, self.D, self.NB = num_q_heads, num_kv_heads, head_dim, num_blocks
        cfg = CwConfig(BLOCK_SIZE, num_blocks, num_q_heads, num_kv_heads, head_dim, max_position, float(rope_theta),
                       recency_window, int(bool(eager_register)), hash_salt, None, None, None, 0, int(index_key_bits))
        self.k_pool = self.v_pool = self.rope_table = None
        if device is not None:
            import torch
            if not torch.cuda.is_available():
                raise RuntimeError("a device context needs CUDA; there is no CPU fallback")
            dev = torch.device(device)
            nbytes = self.lib.cw_pool_bytes(C.byref(cfg))
            if nbytes < 0:
                raise CwError(int(nbytes), "bad configuration")
            # zero-filled once: stale slots of a partially filled block must hold finite values (cacheweaver.h)
            self.k_pool = torch.zeros(nbytes // 2, dtype=torch.bfloat16, device=dev)
            self.v_pool = torch.zeros(nbytes // 2, dtype=torch.bfloat16, device=dev)
            self.rope_table = torch.empty(max_position * head_dim, dtype=torch.float32, device=dev)
            cfg.k_pool, cfg.v_pool, cfg.rope_table = self.k_pool.data_ptr(), self.v_pool.data_ptr(), self.rope_table.data_ptr()
            cfg.device = dev.index or 0
        self.cfg = cfg
        h = C.c_void_p()
        rc = self.lib.cw_create(C.byref(cfg), C.byref(h))
        if rc != CW_OK:
            raise CwError(rc, self.lib.cw_strerror(rc).decode())
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            self.lib.cw_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc):
        if rc == CW_OK:
            return
        msg = self.lib.cw_strerror(rc).decode()
        if rc in (CW_ERR_CUDA, CW_ERR_INVALID):
            msg += ": " + self.lib.cw_last_error(self.h).decode()
        raise (NoSpace if rc == CW_ERR_NO_SPACE else CwError)(rc, msg)

    # ---- ordering ----
    def cw_order(self, doc_ids):
        d = np.ascontiguousarray(doc_ids, dtype=np.int64)
        out = np.empty_like(d)
        depth = C.c_int32()
        self._check(self.lib.cw_order(self.h, _i64p(d), len(d), _i64p(out), C.byref(depth)))
        return out.tolist(), depth.value

    def cw_order_arm(self, arm, doc_ids, doc_tokens=None, query_tokens=None):
        """arm: ARMS name or id.  doc_tokens int32 [num_docs, doc_len], query_tokens int32 [q_len] (exhaustive arm only)."""
        arm = ARMS[arm] if isinstance(arm, str) else int(arm)
        d = np.ascontiguousarray(doc_ids, dtype=np.int64)
        out = np.empty_like(d)
        depth = C.c_int32()
        dt = _np_i32(doc_tokens) if doc_tokens is not None else None
        qt = _np_i32(query_tokens) if query_tokens is not None else None
        self._check(self.lib.cw_order_arm(self.h, arm, _i64p(d), len(d), _i32p(dt) if dt is not None else None,
                                          dt.shape[0] if dt is not None else 0, dt.shape[1] if dt is not None else 0,
                                          _i32p(qt) if qt is not None else None, len(qt) if qt is not None else 0,
                                          _i64p(out), C.byref(depth)))
        return out.tolist(), depth.value

    def cw_predict(self, order):
        d = np.ascontiguousarray(order, dtype=np.int64)
        depth = C.c_int32()
        self._check(self.lib.cw_predict(self.h, _i64p(d), len(d), C.byref(depth)))
        return depth.value

    def cw_observe(self, order):
        d = np.ascontiguousarray(order, dtype=np.int64)
        self._check(self.lib.cw_observe(self.h, _i64p(d), len(d)))

    def cw_mark_stale(self, order, resident_docs):
        d = np.ascontiguousarray(order, dtype=np.int64)
        self._check(self.lib.cw_mark_stale(self.h, _i64p(d), len(d), int(resident_docs)))

    def cw_feedback(self, order, predicted_docs, actual_docs):
        d = np.ascontiguousarray(order, dtype=np.int64)
        self._check(self.lib.cw_feedback(self.h, _i64p(d), len(d), int(predicted_docs), int(actual_docs)))

    def cw_matched_docs(self, doc_ends, n_cached, n_tokens):
        e = _np_i32(doc_ends)
        out = C.c_int32()
        self._check(self.lib.cw_matched_docs(self.h, _i32p(e), len(e), int(n_cached), int(n_tokens), C.byref(out)))
        return out.value

    def cw_feedback_tokens(self, order, predicted_docs, doc_ends, n_cached, n_tokens):
        """cw_feedback with the matched-document count taken by the library from the lookup's n_cached; returns the count."""
        d, e = np.ascontiguousarray(order, dtype=np.int64), _np_i32(doc_ends)
        out = C.c_int32()
        self._check(self.lib.cw_feedback_tokens(self.h, _i64p(d), len(d), int(predicted_docs), _i32p(e), int(n_cached),
                                                int(n_tokens), C.byref(out)))
        return out.value

    # ---- prefix cache ----
    def cw_hash_chain(self, tokens):
        t = _np_i32(tokens)
        out = np.empty(len(t) // BLOCK_SIZE, dtype=np.uint64)
        self._check(self.lib.cw_hash_chain(self.h, _i32p(t), len(t), out.ctypes.data))
        return out

    def cw_lookup(self, tokens, peek_only=False):
        t = _np_i32(tokens)
        n = len(t)
        nc = C.c_int32()
        if peek_only:
            self._check(self.lib.cw_lookup(self.h, _i32p(t), n, 1, None, None, C.byref(nc)))
            return nc.value
        table = np.empty(-(-n // BLOCK_SIZE), dtype=np.int32)
        req = C.c_int64()
        self._check(self.lib.cw_lookup(self.h, _i32p(t), n, 0, C.byref(req), _i32p(table), C.byref(nc)))
        return req.value, table, nc.value

    def cw_release(self, req):
        self._check(self.lib.cw_release(self.h, req))

    def cw_extend(self, req, new_tokens, cap=None):
        """the live request grows by new_tokens; returns its whole block table (numpy int32)."""
        t = _np_i32(new_tokens)
        cap = int(cap) if cap is not None else self.NB
        table = np.empty(cap, dtype=np.int32)
        nb = C.c_int32()
        self._check(self.lib.cw_extend(self.h, req, _i32p(t), len(t), _i32p(table), cap, C.byref(nb)))
        return table[: nb.value].copy()

    def cw_reset(self):
        self._check(self.lib.cw_reset(self.h))

    def cw_admit_batch(self, doc_ids, reorder, doc_tokens, query_tokens, max_blocks=None, out=None):
        """doc_ids int64 [B,k]; doc_tokens int32 [num_docs, doc_len]; query_tokens int32 [B, q_len] (C-contiguous numpy).
        Returns dict(orders, pred, reqs, tables, n_cached, cu, admitted); `out` may carry preallocated arrays."""
        doc_ids = np.ascontiguousarray(doc_ids, dtype=np.int64)
        doc_tokens, query_tokens = _np_i32(doc_tokens), _np_i32(query_tokens)
        B, k = doc_ids.shape
        num_docs, doc_len = doc_tokens.shape
        q_len = query_tokens.shape[1]
        if max_blocks is None:
            max_blocks = -(-(k * doc_len + q_len) // BLOCK_SIZE)
        o = out or {}
        orders = o.get("orders", np.empty((B, k), dtype=np.int64))
        pred = o.get("pred", np.empty(B, dtype=np.int32))
        reqs = o.get("reqs", np.empty(B, dtype=np.int64))
        tables = o.get("tables", np.empty((B, max_blocks), dtype=np.int32))
        nc = o.get("n_cached", np.empty(B, dtype=np.int32))
        cu = o.get("cu", np.empty(B + 1, dtype=np.int32))
        adm = C.c_int32()
        self._check(self.lib.cw_admit_batch(self.h, _i64p(doc_ids), B, k, ARMS[reorder] if isinstance(reorder, str) else int(reorder), _i32p(doc_tokens), num_docs,
                                            doc_len, _i32p(query_tokens), q_len, _i64p(orders), _i32p(pred), _i64p(reqs),
                                            _i32p(tables), max_blocks, _i32p(nc), _i32p(cu), C.byref(adm)))
        return dict(orders=orders, pred=pred, reqs=reqs, tables=tables, n_cached=nc, cu=cu, admitted=adm.value)

    def cw_release_batch(self, reqs):
        r = np.ascontiguousarray(reqs, dtype=np.int64)
        self._check(self.lib.cw_release_batch(self.h, _i64p(r), len(r)))

    def cw_free_list(self):
        out = np.empty(self.NB, dtype=np.int32)
        n = C.c_int32()
        self._check(self.lib.cw_free_list(self.h, _i32p(out), self.NB, C.byref(n)))
        return out[: n.value].tolist()

    def cw_stats(self):
        s = CwStats()
        self._check(self.lib.cw_stats(self.h, C.byref(s)))
        return {n: getattr(s, n) for n, _ in CwStats._fields_}

    def cw_pool_offset(self, block, kv_head, t, d):
        return self.lib.cw_pool_offset(C.byref(self.cfg), block, kv_head, t, d)

    def cw_q_roped_offset(self, s, tok, head, d):
        return self.lib.cw_q_roped_offset(C.byref(self.cfg), s, tok, head, d)

    # ---- device work ----
    @staticmethod
    def _stream():
        import torch
        return torch.cuda.current_stream().cuda_stream

    def cw_append_kv(self, q, k, v, q_roped, d_cu, d_nc, d_tables, max_blocks, B, T):
        self._check(self.lib.cw_append_kv(self.h, q.data_ptr(), k.data_ptr(), v.data_ptr(), q_roped.data_ptr(),
                                          d_cu.data_ptr(), d_nc.data_ptr(), d_tables.data_ptr(), max_blocks, B, T,
                                          self._stream()))

    def cw_attn_work_ints(self, B, T):
        return int(self.lib.cw_attn_work_ints(self.h, int(B), int(T)))

    def cw_prefill_attn(self, q_roped, out, d_cu, d_nc, d_tables, max_blocks, B, T, max_q_len, max_kv_len, d_work,
                        d_kv_len=None):
        """all descriptors are device int32 tensors; d_work: device int32 scratch of cw_attn_work_ints(B, T) ints."""
        self._check(self.lib.cw_prefill_attn(self.h, q_roped.data_ptr(), out.data_ptr(), d_cu.data_ptr(), d_nc.data_ptr(),
                                             d_kv_len.data_ptr() if d_kv_len is not None else None, d_tables.data_ptr(),
                                             max_blocks, B, T, int(max_q_len), int(max_kv_len), d_work.data_ptr(),
                                             self._stream()))

    def cw_attn_schedule(self, d_cu, d_nc, d_tables, max_blocks, B, T, max_q_len, max_kv_len, d_work, d_kv_len=None):
        """first launch of cw_prefill_attn alone: descriptors -> work list (may run before / beside cw_append_kv)."""
        self._check(self.lib.cw_attn_schedule(self.h, d_cu.data_ptr(), d_nc.data_ptr(),
                                              d_kv_len.data_ptr() if d_kv_len is not None else None, d_tables.data_ptr(),
                                              max_blocks, B, T, int(max_q_len), int(max_kv_len), d_work.data_ptr(),
                                              self._stream()))

    def cw_attn_run(self, q_roped, out, d_tables, max_blocks, B, T, d_work):
        """second launch of cw_prefill_attn alone: the attention kernel over the list cw_attn_schedule wrote."""
        self._check(self.lib.cw_attn_run(self.h, q_roped.data_ptr(), out.data_ptr(), d_tables.data_ptr(), max_blocks, B, T,
                                         d_work.data_ptr(), self._stream()))

    def cw_prefill_attn_static(self, q_roped, out, d_cu, d_nc, d_tables, max_blocks, B, T, max_q_len, max_kv_len,
                               d_status=None, d_kv_len=None):
        """cw_prefill_attn without a d_work argument, for callers that may not allocate device memory: the work list sits
        in a 2 MiB array inside the library (one per GPU, shared by all calls: do not let two calls overlap on the GPU).
        Raises CwError(CW_ERR_INVALID) when cw_attn_work_ints(B, T) > STATIC_WORK_INTS.  d_status: optional device int32[4]
        that receives the work header (error flags at [1])."""
        self._check(self.lib.cw_prefill_attn_static(
            self.h, q_roped.data_ptr(), out.data_ptr(), d_cu.data_ptr(), d_nc.data_ptr(),
            d_kv_len.data_ptr() if d_kv_len is not None else None, d_tables.data_ptr(), max_blocks, B, T, int(max_q_len),
            int(max_kv_len), d_status.data_ptr() if d_status is not None else None, self._stream()))

    def cw_prefill_requests_ws_bytes(self, B, T, max_blocks):
        return int(self.lib.cw_prefill_requests_ws_bytes(self.h, B, T, max_blocks))

    def cw_prefill_requests_work_offset(self, B, max_blocks):
        return int(self.lib.cw_prefill_requests_work_offset(self.h, B, max_blocks))

    def cw_prefill_requests(self, reqs, q, k, v, q_roped, out, T, max_blocks, d_ws):
        """reqs: request handles of the wave (numpy int64, batch order); q, k, v, q_roped, out, d_ws: device tensors."""
        r = np.ascontiguousarray(reqs, dtype=np.int64)
        self._check(self.lib.cw_prefill_requests(self.h, _i64p(r), len(r), q.data_ptr(), k.data_ptr(), v.data_ptr(),
                                                 q_roped.data_ptr(), out.data_ptr(), int(T), int(max_blocks),
                                                 d_ws.data_ptr(), self._stream()))

    def cw_gather_kv(self, d_table, n, k_out, v_out):
        self._check(self.lib.cw_gather_kv(self.h, d_table.data_ptr(), n, k_out.data_ptr(), v_out.data_ptr(),
                                          self._stream()))

    def cw_prefill_host_ws_bytes(self, B, T, max_blocks):
        return int(self.lib.cw_prefill_host_ws_bytes(self.h, B, T, max_blocks))

    def cw_prefill_host(self, h_q, h_k, h_v, h_out, h_cu, h_nc, h_tables, max_blocks, B, T, d_ws):
        """h_q/h_k/h_v/h_out: pinned CPU torch tensors (bf16); descriptors: numpy int32; d_ws: device uint8 tensor."""
        h_cu, h_nc, h_tables = _np_i32(h_cu), _np_i32(h_nc), _np_i32(h_tables)
        self._check(self.lib.cw_prefill_host(self.h, h_q.data_ptr(), h_k.data_ptr(), h_v.data_ptr(), h_out.data_ptr(),
                                             _i32p(h_cu), _i32p(h_nc), _i32p(h_tables), max_blocks, B, T,
                                             d_ws.data_ptr(), self._stream()))
