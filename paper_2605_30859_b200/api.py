"""Thin ctypes binding over the C-ABI in include/darts.h (argument marshalling only).

Importing this module loads csrc/libdarts.so and raises if it is missing: there is no CPU or
PyTorch fallback.  torch is used for device memory (workspace, inputs) and streams only.
The raw entry points are available under their C names (`darts_prefill`, `darts_decode_step`,
`darts_select_and_compact`, `darts_rollout`, ...); `Darts` wraps a context with the same verbs.
"""
import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "csrc", "libdarts.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2605_30859_b200.build` "
                      "(there is no fallback path)")
_lib = C.CDLL(LIB_PATH)

OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_KV_POOL_EXHAUSTED, ERR_WORKSPACE_TOO_SMALL, ERR_CUDA, ERR_BAD_STATE = range(7)
F32, BF16 = 0, 1
ROW_ACTIVE, ROW_VALID, ROW_TRUNC, ROW_PRUNED = 0, 1, 2, 3
MODE_AUTO, MODE_DUAL_END, MODE_SHORTEST_EARLY_STOP = 0, 1, 2
FLAG_DUMP_LOGITS, FLAG_NO_PREFIX_SHARING, FLAG_PROFILE_ATTENTION, FLAG_DUMP_HIDDEN, FLAG_LM_HEAD_TILES, FLAG_CTA_PAIRS = 1, 2, 4, 8, 16, 32

_vp, _i32, _u32, _u64, _f32 = C.c_void_p, C.c_int32, C.c_uint32, C.c_uint64, C.c_float
_pp = C.POINTER(C.c_void_p)


class ModelDesc(C.Structure):
    _fields_ = [(n, _i32) for n in ("n_layers", "d_model", "n_q_heads", "n_kv_heads", "head_dim", "ffn", "vocab",
                                    "n_experts", "top_k", "expert_ffn", "dtype", "qk_norm")] + \
               [("rope_theta", _f32), ("rms_eps", _f32), ("eos_id", _i32)]


class Weights(C.Structure):
    _fields_ = [("embed", _vp), ("final_norm", _vp), ("lm_head", _vp)] + \
               [(n, _pp) for n in ("attn_norm", "wqkv", "q_norm", "k_norm", "wo", "mlp_norm", "wgu", "wd", "wr", "wgu_e", "wd_e")]


class RuntimeDesc(C.Structure):
    _fields_ = [(n, _i32) for n in ("page_size", "n_pages", "max_rows", "max_prompts", "max_prompt_len", "max_new",
                                    "prefill_chunk")] + \
               [("flags", _u32), ("workspace", _vp), ("workspace_bytes", C.c_size_t), ("stream", _vp)]


class Policy(C.Structure):
    _fields_ = [("K", _i32), ("L_long", _i32), ("M_up", _i32), ("mode", _i32)]


class Results(C.Structure):
    _fields_ = [(n, _vp) for n in ("tokens", "len", "status", "margin", "sel", "sel_mask", "close_step", "len_mean", "len_var", "logprob", "n_pruned")]


class Counters(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("n_steps", "n_generated_tokens", "n_kept_tokens", "n_near_ties", "n_row_steps",
                                         "peak_pages", "kernel_launches", "pages_allocated")]


def _sig(name, *argtypes, restype=_i32):
    f = getattr(_lib, name)
    f.argtypes, f.restype = list(argtypes), restype
    return f


_ctx = C.c_void_p
darts_workspace_bytes = _sig("darts_workspace_bytes", C.POINTER(ModelDesc), C.POINTER(RuntimeDesc), C.POINTER(C.c_size_t))
darts_create = _sig("darts_create", C.POINTER(ModelDesc), C.POINTER(Weights), C.POINTER(RuntimeDesc), C.POINTER(_ctx))
darts_destroy = _sig("darts_destroy", _ctx)
darts_last_error = _sig("darts_last_error", _ctx, restype=C.c_char_p)
darts_prefill = _sig("darts_prefill", _ctx, _vp, _vp, _i32, _vp, _vp, C.POINTER(Policy), _f32, _u64)
darts_decode_step = _sig("darts_decode_step", _ctx)
darts_select_and_compact = _sig("darts_select_and_compact", _ctx, _vp)
darts_rollout = _sig("darts_rollout", _ctx, _vp, _i32, _i32, _i32, _i32, _i32, _f32, _u64, _vp, C.POINTER(Results))
darts_run_to_completion = _sig("darts_run_to_completion", _ctx, C.POINTER(Results))
ChunkFn = C.CFUNCTYPE(None, C.c_void_p, _i32, _i32, _i32, C.POINTER(C.c_int32), C.POINTER(C.c_float))
darts_run_to_completion_streaming = _sig("darts_run_to_completion_streaming", _ctx, _i32, ChunkFn, C.c_void_p, C.POINTER(Results))
darts_rollout_host = _sig("darts_rollout_host", _ctx, _vp, _i32, _i32, _vp, _vp, C.POINTER(Policy), _i32, _f32, _u64,
                          C.POINTER(Results))
darts_score_begin = _sig("darts_score_begin", _ctx, _vp, _vp, _i32, _vp, _f32)
darts_score_chunk = _sig("darts_score_chunk", _ctx, _i32, _i32, _vp, _vp)
darts_get_results = _sig("darts_get_results", _ctx, C.POINTER(Results))
darts_get_counters = _sig("darts_get_counters", _ctx, C.POINTER(Counters))
darts_n_active = _sig("darts_n_active", _ctx, C.POINTER(_i32))
darts_get_attention_times = _sig("darts_get_attention_times", _ctx, _vp, _i32, C.POINTER(_i32))
darts_debug_logits = _sig("darts_debug_logits", _ctx, _i32, _vp)
darts_debug_routing = _sig("darts_debug_routing", _ctx, _i32, _i32, _vp)
darts_debug_hidden = _sig("darts_debug_hidden", _ctx, _i32, _i32, _i32, _vp)
darts_debug_row_slots = _sig("darts_debug_row_slots", _ctx, _vp, _vp, _i32)
darts_debug_fast_forward = _sig("darts_debug_fast_forward", _ctx, _i32)
darts_debug_set_last_tokens = _sig("darts_debug_set_last_tokens", _ctx, _vp, _i32)
darts_debug_gemm_bf16 = _sig("darts_debug_gemm_bf16", _ctx, _vp, _vp, _vp, _vp, _i32, _i32, _i32, _i32)
darts_debug_gemm_scratch_floats = _sig("darts_debug_gemm_scratch_floats", _ctx, _i32, _i32, _i32, _i32, C.POINTER(C.c_size_t))
darts_static_scratch_bytes = _sig("darts_static_scratch_bytes", C.POINTER(C.c_size_t))
darts_gemm_bf16_static = _sig("darts_gemm_bf16_static", _ctx, _vp, _vp, _vp, _i32, _i32, _i32)
darts_update_variance_ema = _sig("darts_update_variance_ema", _vp, _vp, _i32, _f32)
darts_redundancy_budget = _sig("darts_redundancy_budget", C.c_double, C.c_double, C.c_double, _i32, _i32, C.POINTER(C.c_int64))
darts_allocate_redundancy = _sig("darts_allocate_redundancy", _vp, _i32, C.c_int64, _i32, _i32, _vp)
darts_attn_load = _sig("darts_attn_load", _ctx, _i32, _i32, _i32, _vp, _vp, _vp, _vp, _vp)
darts_attention = _sig("darts_attention", _ctx, _i32, _vp, _vp)


class DartsError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"darts status {code}: {msg}")
        self.code = code


def _np_ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _ptr_array(tensors):
    arr = (C.c_void_p * len(tensors))(*[t.data_ptr() for t in tensors])
    return C.cast(arr, _pp), arr


def model_desc(cfg, eos_id=None):
    m = ModelDesc()
    for k in ("n_layers", "d_model", "n_q_heads", "n_kv_heads", "head_dim", "ffn", "vocab", "n_experts", "top_k", "expert_ffn"):
        setattr(m, k, int(cfg[k]))
    m.dtype = F32 if cfg["dtype"] == "f32" else BF16
    m.qk_norm = int(bool(cfg.get("qk_norm", False)))
    m.rope_theta, m.rms_eps = float(cfg["rope_theta"]), float(cfg["rms_eps"])
    m.eos_id = int(cfg["vocab"] - 1 if eos_id is None else eos_id)
    return m


def update_variance_ema(var_ema, len_var, beta):
    """In-place EMA of the per-prompt length variances (float32 arrays)."""
    assert var_ema.dtype == np.float32 and var_ema.flags.c_contiguous
    lv = np.ascontiguousarray(len_var, dtype=np.float32)
    st = darts_update_variance_ema(_np_ptr(var_ema), _np_ptr(lv), len(var_ema), beta)
    if st != OK:
        raise DartsError(st, "darts_update_variance_ema")
    return var_ema


def redundancy_budget(rho, lam, k, G, K):
    out = C.c_int64()
    st = darts_redundancy_budget(rho, lam, k, G, K, C.byref(out))
    if st != OK:
        raise DartsError(st, "darts_redundancy_budget")
    return out.value


def allocate_redundancy(var_ema, M_total, M_low, M_up):
    v = np.ascontiguousarray(var_ema, dtype=np.float32)
    out = np.empty(len(v), np.int32)
    st = darts_allocate_redundancy(_np_ptr(v), len(v), M_total, M_low, M_up, _np_ptr(out))
    if st != OK:
        raise DartsError(st, "darts_allocate_redundancy")
    return out


class Darts:
    """One context = one GPU = one stream.  `model` is the dict built by workloads.make_model(device='cuda')
    (tensors are borrowed: keep the dict alive), or just {'cfg': ...} for an attention-only context."""

    def __init__(self, model, page_size, n_pages, max_rows, max_prompts, max_prompt_len, max_new, flags=0,
                 prefill_chunk=0, eos_id=None, stream=None):
        self.model, self.cfg = model, model["cfg"]
        self.m = model_desc(self.cfg, eos_id)
        self._keep = []
        w = None
        if self.cfg["vocab"] > 0:
            w = Weights()
            w.embed, w.final_norm, w.lm_head = (model[k].data_ptr() for k in ("embed", "final_norm", "lm_head"))
            for name in ("attn_norm", "wqkv", "q_norm", "k_norm", "wo", "mlp_norm", "wgu", "wd", "wr", "wgu_e", "wd_e"):
                if name in model["layers"][0]:
                    p, arr = _ptr_array([L[name] for L in model["layers"]])
                    self._keep.append(arr)
                    setattr(w, name, p)
        rt = RuntimeDesc(page_size=page_size, n_pages=n_pages, max_rows=max_rows, max_prompts=max_prompts,
                         max_prompt_len=max_prompt_len, max_new=max_new, prefill_chunk=prefill_chunk, flags=flags)
        need = C.c_size_t()
        st = darts_workspace_bytes(C.byref(self.m), C.byref(rt), C.byref(need))
        if st != OK:
            raise DartsError(st, "darts_workspace_bytes rejected the descriptors")
        self.workspace = torch.empty(need.value, dtype=torch.uint8, device="cuda")
        self.stream = torch.cuda.current_stream() if stream is None else stream
        rt.workspace, rt.workspace_bytes, rt.stream = self.workspace.data_ptr(), need.value, self.stream.cuda_stream
        self.rt = rt
        self.ctx = _ctx()
        st = darts_create(C.byref(self.m), C.byref(w) if w is not None else None, C.byref(rt), C.byref(self.ctx))
        if st != OK:
            msg = darts_last_error(self.ctx).decode() if self.ctx else "darts_create failed"
            if self.ctx:
                darts_destroy(self.ctx)
                self.ctx = None
            raise DartsError(st, msg)
        self.G = self.R = self.K = 0
        self.max_new = max_new

    def close(self):
        if getattr(self, "ctx", None):
            darts_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        self.close()

    def _check(self, st):
        if st != OK:
            raise DartsError(st, darts_last_error(self.ctx).decode())

    # ---- the four verbs of the path -------------------------------------------------------------
    def prefill(self, prompts, Kp, K, temperature=1.0, seed=0, forced_len=None, L_long=1, M_up=0, mode=MODE_AUTO):
        """prompts: list of int arrays (ragged) or [G,P] array; Kp: [G]; forced_len: [G, max Kp] or None."""
        plist = [np.asarray(p, dtype=np.int32) for p in prompts]
        G = len(plist)
        offs = np.concatenate([[0], np.cumsum([len(p) for p in plist])]).astype(np.int32)
        toks = torch.from_numpy(np.concatenate(plist)).cuda()
        Kp = np.ascontiguousarray(Kp, dtype=np.int32)
        fl = None
        if forced_len is not None:
            fl = torch.from_numpy(np.ascontiguousarray(forced_len, dtype=np.int32)).cuda()
            assert fl.shape == (G, int(Kp.max()))
        pol = Policy(K=K, L_long=L_long, M_up=M_up, mode=mode)
        self._check(darts_prefill(self.ctx, toks.data_ptr(), _np_ptr(offs), G, _np_ptr(Kp), fl.data_ptr() if fl is not None else None,
                                  C.byref(pol), temperature, seed))
        self.G, self.R, self.K = G, int(Kp.sum()), K
        self._keep_inputs = (toks, fl)

    def prefill_device(self, prompts_dev, P, Kp, K, temperature=1.0, seed=0, forced_len_dev=None, L_long=1, M_up=0, mode=MODE_AUTO,
                       max_len=None):
        """darts_prefill with inputs already resident in HBM: prompts_dev [G,P] int32 (cuda), forced_len_dev [G, max Kp] int32 (cuda)."""
        assert prompts_dev.is_cuda and prompts_dev.dtype == torch.int32 and prompts_dev.is_contiguous()
        assert max_len is None or max_len == self.max_new
        G = prompts_dev.shape[0]
        Kp = np.ascontiguousarray(Kp, dtype=np.int32)
        offs = (np.arange(G + 1) * P).astype(np.int32)
        if forced_len_dev is not None:
            assert forced_len_dev.is_cuda and forced_len_dev.dtype == torch.int32 and tuple(forced_len_dev.shape) == (G, int(Kp.max()))
        pol = Policy(K=K, L_long=L_long, M_up=M_up, mode=mode)
        self._check(darts_prefill(self.ctx, prompts_dev.data_ptr(), _np_ptr(offs), G, _np_ptr(Kp),
                                  forced_len_dev.data_ptr() if forced_len_dev is not None else None, C.byref(pol), temperature, seed))
        self.G, self.R, self.K = G, int(Kp.sum()), K
        self._keep_inputs = (prompts_dev, forced_len_dev)

    def decode_step(self):
        self._check(darts_decode_step(self.ctx))

    def select_and_compact(self):
        self._check(darts_select_and_compact(self.ctx, None))

    def n_active(self):
        n = _i32()
        self._check(darts_n_active(self.ctx, C.byref(n)))
        return n.value

    def run_to_completion(self):
        self._check(darts_run_to_completion(self.ctx, None))

    def run_to_completion_streaming(self, chunk_steps, on_chunk):
        """on_chunk(step_begin, step_end, tokens, logprob): int32 / float32 numpy arrays [n_rows, step_end - step_begin] (copied)."""
        def tramp(_user, s0, s1, n_rows, ptr, lp):
            on_chunk(s0, s1, np.ctypeslib.as_array(ptr, shape=(n_rows, s1 - s0)).copy(), np.ctypeslib.as_array(lp, shape=(n_rows, s1 - s0)).copy())
        cb = ChunkFn(tramp)
        self._check(darts_run_to_completion_streaming(self.ctx, chunk_steps, cb, None, None))

    # ---- consumer side of token-level streaming ------------------------------------------------------
    def score_begin(self, prompts, Kp, temperature=1.0):
        """Prefill the prompts (list of int arrays or [G,P]) for chunk scoring: no sampling, rows = sum Kp."""
        plist = [np.asarray(p, dtype=np.int32) for p in prompts]
        offs = np.concatenate([[0], np.cumsum([len(p) for p in plist])]).astype(np.int32)
        toks = torch.from_numpy(np.concatenate(plist)).cuda()
        Kp = np.ascontiguousarray(Kp, dtype=np.int32)
        self._check(darts_score_begin(self.ctx, toks.data_ptr(), _np_ptr(offs), len(plist), _np_ptr(Kp), temperature))
        self.G, self.R = len(plist), int(Kp.sum())

    def score_chunk(self, step_begin, step_end, tokens):
        """tokens int32 [n_rows, step_end - step_begin] (-1 from a row's end on) -> float32 log-probabilities, same shape."""
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        assert t.shape == (self.R, step_end - step_begin)
        out = np.empty(t.shape, np.float32)
        self._check(darts_score_chunk(self.ctx, step_begin, step_end, _np_ptr(t), _np_ptr(out)))
        return out

    def rollout(self, prompts_dev, G, Kp, K, max_len, temperature, seed, forced_len_dev=None, fetch=True):
        """north_star signature: device prompts [G,P] int32, scalar K' (L_long = 1, M_up = 2K, mode AUTO); forced_len_dev [G,K'] int32
        (cuda) or None.  fetch=True hands darts_rollout a darts_results and returns its buffers; False passes out = NULL."""
        assert prompts_dev.is_cuda and prompts_dev.dtype == torch.int32 and prompts_dev.is_contiguous()
        assert forced_len_dev is None or (forced_len_dev.is_cuda and forced_len_dev.dtype == torch.int32 and tuple(forced_len_dev.shape) == (G, Kp))
        self.G, self.R, self.K = G, G * Kp, K
        bufs, res = self._result_buffers() if fetch else (None, None)
        self._check(darts_rollout(self.ctx, prompts_dev.data_ptr(), prompts_dev.shape[1], G, Kp, K, max_len, temperature, seed,
                                  forced_len_dev.data_ptr() if forced_len_dev is not None else None, C.byref(res) if fetch else None))
        return bufs

    def rollout_host(self, prompts, Kp, K, max_len, temperature, seed, forced_len=None, L_long=1, M_up=0, mode=MODE_AUTO,
                     out=None):
        """HOST inputs -> HOST results in one call (prompts [G,P] int32 numpy, Kp [G])."""
        prompts = np.ascontiguousarray(prompts, dtype=np.int32)
        Kp = np.ascontiguousarray(Kp, dtype=np.int32)
        G, P = prompts.shape
        fl = None if forced_len is None else np.ascontiguousarray(forced_len, dtype=np.int32)
        pol = Policy(K=K, L_long=L_long, M_up=M_up, mode=mode)
        self.G, self.R, self.K = G, int(Kp.sum()), K
        bufs, res = self._result_buffers() if out is None else out
        self._check(darts_rollout_host(self.ctx, _np_ptr(prompts), P, G, _np_ptr(Kp), _np_ptr(fl) if fl is not None else None,
                                       C.byref(pol), max_len, temperature, seed, C.byref(res)))
        return bufs

    # ---- read-back ------------------------------------------------------------------------------
    def _result_buffers(self):
        R, G, K, mn = self.R, self.G, self.K, self.max_new
        bufs = dict(tokens=np.empty((R, mn), np.int32), len=np.empty(R, np.int32), status=np.empty(R, np.uint8),
                    margin=np.empty((R, mn), np.float32), sel=np.empty((G, K), np.int32), sel_mask=np.empty(G, np.uint32),
                    close_step=np.empty(G, np.int32), len_mean=np.empty(G, np.float32), len_var=np.empty(G, np.float32),
                    logprob=np.empty((R, mn), np.float32), n_pruned=np.empty(G, np.int32))
        res = Results(**{k: _np_ptr(v) for k, v in bufs.items()})
        return bufs, res

    def results(self):
        bufs, res = self._result_buffers()
        self._check(darts_get_results(self.ctx, C.byref(res)))
        return bufs

    def counters(self):
        c = Counters()
        self._check(darts_get_counters(self.ctx, C.byref(c)))
        return {n: getattr(c, n) for n, _ in Counters._fields_}

    def attention_times(self):
        """ms per decode step of layer 0's attention launches (needs FLAG_PROFILE_ATTENTION)."""
        n = _i32()
        self._check(darts_get_attention_times(self.ctx, None, 0, C.byref(n)))
        out = np.empty(n.value, np.float32)
        if n.value:
            self._check(darts_get_attention_times(self.ctx, _np_ptr(out), n.value, C.byref(n)))
        return out

    def debug_logits(self, row):
        out = np.empty(self.cfg["vocab"], np.float32)
        self._check(darts_debug_logits(self.ctx, row, _np_ptr(out)))
        return out

    def debug_routing(self, slot_begin, n_slots):
        """Expert ids [n_layers, n_slots, top_k] the routers chose for a slot range of the most recent pass (MoE + FLAG_DUMP_LOGITS)."""
        out = np.empty((self.cfg["n_layers"], n_slots, self.cfg["top_k"]), np.int32)
        self._check(darts_debug_routing(self.ctx, slot_begin, n_slots, _np_ptr(out)))
        return out

    def debug_hidden(self, slot_begin, n_slots):
        """fp32 residual stream [n_layers + 1, n_slots, d_model] at every layer boundary of the most recent pass (FLAG_DUMP_HIDDEN)."""
        out = np.empty((self.cfg["n_layers"] + 1, n_slots, self.cfg["d_model"]), np.float32)
        for b in range(self.cfg["n_layers"] + 1):
            self._check(darts_debug_hidden(self.ctx, b, slot_begin, n_slots, _np_ptr(out[b])))
        return out

    def debug_row_slots(self):
        """(slot, step) of every row's last decode step."""
        slot, step = np.empty(self.R, np.int32), np.empty(self.R, np.int32)
        self._check(darts_debug_row_slots(self.ctx, _np_ptr(slot), _np_ptr(step), self.R))
        return slot, step

    def debug_fast_forward(self, new_len):
        """Profiling hook: every active row gets a generated length of new_len (KV of the skipped positions is not computed)."""
        self._check(darts_debug_fast_forward(self.ctx, new_len))

    def debug_set_last_tokens(self, tokens):
        t = np.ascontiguousarray(tokens, dtype=np.int32)
        self._check(darts_debug_set_last_tokens(self.ctx, _np_ptr(t), len(t)))

    def debug_gemm_bf16(self, X, W, split_k=1, scratch=None, reduce=True):
        """C = X @ W.T on the tcgen05 GEMM (bf16 device tensors X [rows,K], W [N,K]); returns fp32 [rows,N] on device
        (reduce=False: only the split-K partials are computed, into `scratch`)."""
        rows, K = X.shape
        N = W.shape[0]
        out = torch.empty(rows, N, dtype=torch.float32, device="cuda") if reduce else None
        if scratch is None:
            need = C.c_size_t()
            self._check(darts_debug_gemm_scratch_floats(self.ctx, rows, N, K, split_k, C.byref(need)))
            scratch = torch.empty(need.value, dtype=torch.float32, device="cuda")
        self._check(darts_debug_gemm_bf16(self.ctx, X.data_ptr(), W.data_ptr(), out.data_ptr() if reduce else None, scratch.data_ptr(),
                                          rows, N, K, split_k))
        self._scratch = scratch
        return out if reduce else scratch

    def gemm_bf16_static(self, X, W, out):
        """out[rows,N] (fp32, device, caller-allocated) = X @ W.T on the stream-K GEMM with its pieces in the library's static device
        scratch (darts_gemm_bf16_static): nothing is allocated by this call.  Raises DartsError(ERR_WORKSPACE_TOO_SMALL) beyond the limit."""
        rows, K = X.shape
        N = W.shape[0]
        assert out.shape == (rows, N) and out.dtype == torch.float32 and out.is_contiguous() and X.is_contiguous() and W.is_contiguous()
        self._check(darts_gemm_bf16_static(self.ctx, X.data_ptr(), W.data_ptr(), out.data_ptr(), rows, N, K))
        return out

    # ---- attention-only (config 2) -----------------------------------------------------------------
    def attn_load(self, G, P, Kp, k_prefix, v_prefix, suffix_len, k_suffix, v_suffix):
        sl = np.ascontiguousarray(suffix_len, dtype=np.int32)
        self._check(darts_attn_load(self.ctx, G, P, Kp, k_prefix.data_ptr(), v_prefix.data_ptr(), _np_ptr(sl),
                                    k_suffix.data_ptr(), v_suffix.data_ptr()))
        self.G, self.R = G, G * Kp

    def attention(self, q, out, layer=0):
        self._check(darts_attention(self.ctx, layer, q.data_ptr(), out.data_ptr()))
