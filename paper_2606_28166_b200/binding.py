"""ctypes binding over libtandem.so (include/tandem.h). Argument marshalling only - every step of the
path runs in the library's CUDA kernels. No CPU fallback: compute calls raise if the library is missing."""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
lib_path = os.path.join(HERE, "libtandem.so")

SENIOR, JUNIOR, DRAW = 0, 1, 2
TOGGLE, REDRAW = 0, 1
F32, BF16 = 0, 1
GEMM_AUTO, GEMM_SIMT, GEMM_TCGEN05 = 0, 1, 2
ATTN_AUTO, ATTN_ALU, ATTN_MMA = 0, 1, 2
_ERR = {0: "OK", -1: "EINVAL", -2: "ENOMEM", -3: "ECUDA", -4: "ESTATE", -5: "EFULL"}

EXPORTED_SYMBOLS = ["tandem_init", "tandem_load_weights", "tandem_step", "tandem_generate", "tandem_score", "tandem_grpo_objective", "tandem_grpo_objective_static", "tandem_reset",
                    "tandem_free", "tandem_last_error", "tandem_get_stats", "tandem_evict", "tandem_set_profile", "tandem_get_profile",
                    "tandem_kernel_class_name", "tandem_test_set_option", "tandem_test_set_page_order", "tandem_test_uniforms", "tandem_test_nucleus", "tandem_test_philox",
                    "tandem_test_gemm", "tandem_test_gemm_time"]
KC_NUM = 17


class TandemError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__(f"tandem error {_ERR.get(code, code)}: {msg}")
        self.code = code


class _Config(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "hidden", "n_q_heads", "n_kv_heads", "head_dim", "intermediate", "vocab")] + \
               [("rms_eps", C.c_float), ("rope_theta", C.c_float), ("dtype", C.c_int32), ("page_tokens", C.c_int32),
                ("max_seqs", C.c_int32), ("max_seq_len", C.c_int32), ("kv_bytes_per_model", C.c_int64), ("device", C.c_int32),
                ("max_rows_per_step", C.c_int32), ("gemm_impl", C.c_int32), ("use_graph", C.c_int32), ("attn_impl", C.c_int32), ("share_prompt_pages", C.c_int32), ("reserved", C.c_int32 * 2)]


_PP = C.POINTER(C.c_void_p)


class _Weights(C.Structure):
    _fields_ = [("embed", C.c_void_p), ("lm_head", C.c_void_p), ("final_norm", C.c_void_p),
                ("attn_norm", _PP), ("wq", _PP), ("wk", _PP), ("wv", _PP), ("wo", _PP), ("mlp_norm", _PP),
                ("w_gate", _PP), ("w_up", _PP), ("w_down", _PP), ("on_device", C.c_int32)]


class _Params(C.Structure):
    _fields_ = [("p", C.c_float), ("switch_mode", C.c_int32), ("start_owner", C.c_int32), ("cap_k", C.c_int32),
                ("temperature", C.c_float), ("top_p", C.c_float), ("top_k", C.c_int32), ("eos_id", C.c_int32), ("seed", C.c_uint64),
                ("word_start", C.c_void_p)]


class _Overrides(C.Structure):
    _fields_ = [("forced_tokens", C.c_void_p), ("forced_stride", C.c_int64), ("u_switch", C.c_void_p), ("u_switch_stride", C.c_int64),
                ("u_sample", C.c_void_p), ("u_sample_stride", C.c_int64), ("dbg_logits", C.c_void_p)]


class _StepIn(C.Structure):
    _fields_ = [("params", C.POINTER(_Params)), ("n_admit", C.c_int32), ("admit_tokens", C.c_void_p), ("admit_offsets", C.c_void_p),
                ("admit_seq_id", C.c_void_p), ("admit_max_new", C.c_void_p), ("ovr", C.POINTER(_Overrides))]


class _StepOut(C.Structure):
    _fields_ = [("token", C.c_void_p), ("owner", C.c_void_p), ("sen_logp", C.c_void_p), ("done", C.c_void_p), ("argmax", C.c_void_p),
                ("n_active", C.c_void_p), ("admit_slots", C.c_void_p)]


class _Stats(C.Structure):
    _fields_ = [(n, C.c_int64) for n in ("steps", "tokens_emitted", "rows_senior", "rows_junior", "catchup_rows", "kv_bytes_read", "weight_bytes_read")] + \
               [("peak_pages_senior", C.c_int32), ("peak_pages_junior", C.c_int32), ("peak_resident", C.c_int32), ("seconds_total", C.c_double),
                ("kernel_launches", C.c_int64), ("shared_prompt_rows", C.c_int64), ("starved", C.c_int64), ("preemptions", C.c_int64),
                ("kv_bytes_shared_reads", C.c_int64)]


_lib = None


def lib():
    """The loaded shared library. Raises (loudly) if it has not been built: there is no fallback path."""
    global _lib
    if _lib is None:
        if not os.path.exists(lib_path):
            raise TandemError(-4, f"{lib_path} is missing: run `python -m paper_2606_28166_b200.build` (or __graft_entry__.build())")
        L = C.CDLL(lib_path)
        L.tandem_init.argtypes = [C.POINTER(_Config), C.POINTER(C.c_void_p)]
        L.tandem_load_weights.argtypes = [C.c_void_p, C.c_int, C.POINTER(_Weights)]
        L.tandem_step.argtypes = [C.c_void_p, C.POINTER(_StepIn), C.POINTER(_StepOut), C.c_void_p]
        L.tandem_score.argtypes = [C.c_void_p, C.c_int32, C.c_void_p, C.c_void_p, C.c_float, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tandem_grpo_objective.argtypes = [C.c_int32, C.c_int32, C.c_int32] + [C.c_void_p] * 6 + [C.c_float] * 3 + [C.c_void_p] * 5
        L.tandem_grpo_objective_static.argtypes = [C.c_int32, C.c_int32, C.c_int32] + [C.c_void_p] * 6 + [C.c_float] * 3 + [C.c_void_p] * 3
        L.tandem_generate.argtypes = [C.c_void_p, C.POINTER(_Params), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.POINTER(_Overrides), C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p,
                                      C.POINTER(_Stats), C.c_void_p]
        L.tandem_reset.argtypes = [C.c_void_p]
        L.tandem_evict.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
        L.tandem_get_stats.argtypes = [C.c_void_p, C.POINTER(_Stats)]
        L.tandem_set_profile.argtypes = [C.c_void_p, C.c_int]
        L.tandem_get_profile.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
        L.tandem_kernel_class_name.argtypes = [C.c_int]
        L.tandem_kernel_class_name.restype = C.c_char_p
        L.tandem_free.argtypes = [C.c_void_p]
        L.tandem_free.restype = None
        L.tandem_last_error.argtypes = [C.c_void_p]
        L.tandem_last_error.restype = C.c_char_p
        L.tandem_test_uniforms.argtypes = [C.c_uint64, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p]
        L.tandem_test_nucleus.argtypes = [C.c_int32, C.c_float, C.c_float, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tandem_test_philox.argtypes = [C.POINTER(C.c_uint32), C.POINTER(C.c_uint32), C.POINTER(C.c_uint32)]
        L.tandem_test_gemm.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p]
        L.tandem_test_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_int32]
        L.tandem_test_set_page_order.argtypes = [C.c_void_p, C.c_uint64]
        L.tandem_test_gemm_time.argtypes = [C.c_int32] * 7 + [C.POINTER(C.c_float)]
        _lib = L
    return _lib


class TandemConfig:
    """Mirror of tandem_config. `shape` is any object with the model dimensions (e.g. workloads.ModelShape)."""

    def __init__(self, shape, max_seqs, max_seq_len, kv_bytes_per_model=0, device=0, max_rows_per_step=0,
                 gemm_impl=GEMM_AUTO, use_graph=0, page_tokens=16, attn_impl=ATTN_AUTO, share_prompt_pages=0):
        self.shape = shape
        self.c = _Config(shape.n_layers, shape.hidden, shape.n_q_heads, shape.n_kv_heads, shape.head_dim, shape.intermediate,
                         shape.vocab, shape.rms_eps, shape.rope_theta, F32 if shape.dtype == "f32" else BF16, page_tokens,
                         max_seqs, max_seq_len, kv_bytes_per_model, device, max_rows_per_step, gemm_impl, use_graph, attn_impl,
                         share_prompt_pages)


class TandemParams:
    """Mirror of tandem_params; `word_start` is a uint8 NumPy array [vocab] (host)."""

    def __init__(self, word_start, p=0.5, switch_mode=TOGGLE, start_owner=SENIOR, cap_k=0, temperature=1.0, top_p=1.0,
                 eos_id=-1, seed=0, top_k=0):
        self.word_start = np.ascontiguousarray(word_start, dtype=np.uint8)
        self.c = _Params(p, switch_mode, start_owner, cap_k, temperature, top_p, top_k, eos_id, seed, self.word_start.ctypes.data)


def _ptr(t):
    """Device/host pointer of a torch tensor or NumPy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        return t.ctypes.data
    return t.data_ptr()


def _overrides(forced_tokens=None, u_switch=None, u_sample=None, dbg_logits=None):
    if forced_tokens is None and u_switch is None and u_sample is None and dbg_logits is None:
        return None, None
    o = _Overrides(_ptr(forced_tokens), forced_tokens.shape[1] if forced_tokens is not None else 0,
                   _ptr(u_switch), u_switch.shape[1] if u_switch is not None else 0,
                   _ptr(u_sample), u_sample.shape[1] if u_sample is not None else 0, _ptr(dbg_logits))
    return o, (forced_tokens, u_switch, u_sample, dbg_logits)   # keep the tensors alive


class Tandem:
    """Handle owner. Methods carry the names of the C calls: load_weights, step, generate, reset, free."""

    def __init__(self, config):
        self.config = config
        self._h = C.c_void_p()
        rc = lib().tandem_init(C.byref(config.c), C.byref(self._h))
        if rc:
            raise TandemError(rc, "tandem_init failed (see stderr)")

    def _check(self, rc):
        if rc:
            raise TandemError(rc, lib().tandem_last_error(self._h).decode())

    def load_weights(self, model, w):
        """w: dict as produced by workloads.make_weights (torch tensors on CPU or CUDA, dtype matching the config)."""
        L = len(w["layers"])
        keep = []

        def arr(name):
            a = (C.c_void_p * L)(*[w["layers"][l][name].data_ptr() for l in range(L)])
            keep.append(a)
            return C.cast(a, _PP)

        on_dev = 1 if w["embed"].is_cuda else 0
        for t in [w["embed"], w["lm_head"], w["final_norm"]] + [v for l in w["layers"] for v in l.values()]:
            assert t.is_contiguous() and bool(t.is_cuda) == bool(on_dev)
        cw = _Weights(w["embed"].data_ptr(), w["lm_head"].data_ptr(), w["final_norm"].data_ptr(), arr("attn_norm"), arr("wq"),
                      arr("wk"), arr("wv"), arr("wo"), arr("mlp_norm"), arr("w_gate"), arr("w_up"), arr("w_down"), on_dev)
        self._check(lib().tandem_load_weights(self._h, model, C.byref(cw)))

    def step(self, params, admit=None, out=None, forced_tokens=None, u_switch=None, u_sample=None, dbg_logits=None, stream=None):
        """One engine step. admit = (prompts list of int32 arrays, seq_ids or None, max_new int32 array) or None.
        out = dict of optional device tensors: token, owner, sen_logp, done, argmax, n_active. Returns admitted slots."""
        o, keep = _overrides(forced_tokens, u_switch, u_sample, dbg_logits)
        si = _StepIn(C.pointer(params.c), 0, None, None, None, None, C.pointer(o) if o is not None else None)
        slots = None
        if admit is not None:
            prompts, seq_ids, max_new = admit
            toks = np.ascontiguousarray(np.concatenate(prompts), dtype=np.int32)
            offs = np.zeros(len(prompts) + 1, dtype=np.int64)
            offs[1:] = np.cumsum([len(p) for p in prompts])
            mx = np.ascontiguousarray(max_new, dtype=np.int32)
            ids = None if seq_ids is None else np.ascontiguousarray(seq_ids, dtype=np.int32)
            slots = np.zeros(len(prompts), dtype=np.int32)
            si.n_admit = len(prompts); si.admit_tokens = toks.ctypes.data; si.admit_offsets = offs.ctypes.data
            si.admit_seq_id = _ptr(ids); si.admit_max_new = mx.ctypes.data
        out = out or {}
        so = _StepOut(_ptr(out.get("token")), _ptr(out.get("owner")), _ptr(out.get("sen_logp")), _ptr(out.get("done")),
                      _ptr(out.get("argmax")), _ptr(out.get("n_active")), _ptr(slots))
        self._check(lib().tandem_step(self._h, C.byref(si), C.byref(so), stream))
        return slots

    def generate(self, params, prompts, max_new, seq_ids=None, forced_tokens=None, u_switch=None, u_sample=None, stream=None):
        """Whole rollouts with host buffers. Returns dict(tokens [B,L] int32, owner [B,L] uint8 (0 senior, 1 junior),
        mask [B,L] uint8 (1 = senior-emitted, valid positions only), sen_logp [B,L] float32, len [B] int32, stats dict)."""
        B = len(prompts)
        toks = np.ascontiguousarray(np.concatenate(prompts), dtype=np.int32) if B else np.zeros(0, np.int32)
        offs = np.zeros(B + 1, dtype=np.int64)
        offs[1:] = np.cumsum([len(p) for p in prompts])
        mx = np.ascontiguousarray(max_new, dtype=np.int32)
        L = int(mx.max()) if B else 1
        ids = None if seq_ids is None else np.ascontiguousarray(seq_ids, dtype=np.int32)
        out_t = np.zeros((B, L), np.int32); out_o = np.zeros((B, L), np.uint8); out_p = np.zeros((B, L), np.float32)
        out_n = np.zeros(B, np.int32)
        st = _Stats()
        o, keep = _overrides(forced_tokens, u_switch, u_sample, None)
        self._check(lib().tandem_generate(self._h, C.byref(params.c), B, toks.ctypes.data, offs.ctypes.data, mx.ctypes.data, _ptr(ids),
                                          C.pointer(o) if o is not None else None, L, out_t.ctypes.data, out_o.ctypes.data,
                                          out_p.ctypes.data, out_n.ctypes.data, C.byref(st), stream))
        valid = np.arange(L)[None, :] < out_n[:, None]
        stats = {n: getattr(st, n) for n, _ in _Stats._fields_}
        return dict(tokens=out_t, owner=out_o, mask=((out_o == 0) & valid).astype(np.uint8), sen_logp=out_p, len=out_n, stats=stats)

    def score(self, streams, temperature=1.0, stream=None):
        """Teacher-forced dual scoring of finished token streams (prompt + response). Returns dict(sen_logp, jun_logp, overlap:
        lists of float32 arrays, one per stream, entry 0 = 0; stats dict). The junior's cross-entropy over a set of positions is
        the mean of -jun_logp there; alpha is the mean of overlap."""
        B = len(streams)
        toks = np.ascontiguousarray(np.concatenate(streams), dtype=np.int32) if B else np.zeros(0, np.int32)
        offs = np.zeros(B + 1, dtype=np.int64)
        offs[1:] = np.cumsum([len(p) for p in streams])
        outs = [np.zeros(max(1, toks.size), np.float32) for _ in range(3)]
        st = _Stats()
        self._check(lib().tandem_score(self._h, B, toks.ctypes.data, offs.ctypes.data, float(temperature), outs[0].ctypes.data,
                                       outs[1].ctypes.data, outs[2].ctypes.data, C.byref(st), stream))
        cut = lambda a: [a[offs[b]:offs[b + 1]].copy() for b in range(B)]
        return dict(sen_logp=cut(outs[0]), jun_logp=cut(outs[1]), overlap=cut(outs[2]), stats={n: getattr(st, n) for n, _ in _Stats._fields_})

    def reset(self):
        self._check(lib().tandem_reset(self._h))

    def evict(self, slot, stream=None):
        """Remove the sequence in `slot` (pages back to the pools, slot free): resolves a stall / dead lock for tandem_step callers."""
        self._check(lib().tandem_evict(self._h, int(slot), stream))

    def get_stats(self):
        st = _Stats()
        self._check(lib().tandem_get_stats(self._h, C.byref(st)))
        return {n: getattr(st, n) for n, _ in _Stats._fields_}

    def set_profile(self, enable):
        self._check(lib().tandem_set_profile(self._h, 1 if enable else 0))

    def set_option(self, name, value):
        """A/B knob for measurements (tandem_test.h: tandem_test_set_option)."""
        self._check(lib().tandem_test_set_option(self._h, name.encode(), int(value)))

    def set_page_order(self, seed):
        """Test hook: hand KV pages out in a seeded pseudo-random order from the next reset on (0 = ascending)."""
        self._check(lib().tandem_test_set_page_order(self._h, int(seed)))

    def get_profile(self):
        """dict kernel class name -> (device milliseconds, launches) accumulated while profiling was enabled."""
        ms = (C.c_double * KC_NUM)(); n = (C.c_int64 * KC_NUM)()
        self._check(lib().tandem_get_profile(self._h, ms, n))
        return {lib().tandem_kernel_class_name(i).decode(): (ms[i], n[i]) for i in range(KC_NUM)}

    def free(self):
        if self._h:
            lib().tandem_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def grpo_objective(rewards, group, lengths, owner, logp_new, logp_old, logp_ref=None, clip_eps=0.2, kl_beta=0.0, adv_eps=1e-6,
                   want_tokens=True, stream=None):
    """Senior-masked GRPO objective on device tensors (torch, CUDA): rewards [B] f32, lengths [B] i32, owner [B, L] u8, logp_* [B, L]
    f32. Returns dict(advantages [B], token_obj [B, L] | None, seq_obj [B], loss, clip_frac, n_senior, n_live) - the scalars after a
    synchronising copy."""
    import torch
    B, L = owner.shape
    assert B % group == 0 and rewards.numel() == B and lengths.numel() == B
    for t_ in (rewards, lengths, owner, logp_new, logp_old) + ((logp_ref,) if logp_ref is not None else ()):
        assert t_.is_cuda and t_.is_contiguous()
    adv = torch.empty(B, dtype=torch.float32, device=owner.device); seq = torch.empty_like(adv)
    tok = torch.empty(B, L, dtype=torch.float32, device=owner.device) if want_tokens else None
    res = torch.empty(8, dtype=torch.float32, device=owner.device)
    rc = lib().tandem_grpo_objective(B // group, group, L, rewards.data_ptr(), lengths.data_ptr(), owner.data_ptr(), logp_new.data_ptr(),
                                     logp_old.data_ptr(), _ptr(logp_ref), clip_eps, kl_beta, adv_eps, adv.data_ptr(), _ptr(tok), seq.data_ptr(),
                                     res.data_ptr(), stream)
    if rc:
        raise TandemError(rc)
    r = res.cpu().numpy()
    return dict(advantages=adv, token_obj=tok, seq_obj=seq, loss=float(r[0]), clip_frac=float(r[1]), n_senior=int(r[2]), n_live=int(r[3]))


GRPO_STATIC_MAX_ROLLOUTS = 8192          # TANDEM_GRPO_STATIC_MAX_ROLLOUTS in include/tandem.h


def grpo_objective_static(rewards, group, lengths, owner, logp_new, logp_old, logp_ref=None, clip_eps=0.2, kl_beta=0.0, adv_eps=1e-6,
                          token_obj=None, result=None, stream=None):
    """tandem_grpo_objective_static: the same objective with the kernel's scratch in the library's static device array - the call
    allocates nothing. `result` (4 floats, CUDA) and `token_obj` ([B, L] floats, CUDA, optional) are the caller's; when `result` is
    None one is made here (that allocation is the binding's convenience, not the entry point's). Returns dict(loss, clip_frac,
    n_senior, n_live, result, token_obj) - the scalars after a synchronising copy. Calls that overlap on the GPU race on the array."""
    import torch
    B, L = owner.shape
    assert B % group == 0 and rewards.numel() == B and lengths.numel() == B
    for t_ in (rewards, lengths, owner, logp_new, logp_old) + ((logp_ref,) if logp_ref is not None else ()):
        assert t_.is_cuda and t_.is_contiguous()
    if result is None:
        result = torch.empty(4, dtype=torch.float32, device=owner.device)
    assert result.is_cuda and result.dtype == torch.float32 and result.numel() >= 4
    rc = lib().tandem_grpo_objective_static(B // group, group, L, rewards.data_ptr(), lengths.data_ptr(), owner.data_ptr(), logp_new.data_ptr(),
                                            logp_old.data_ptr(), _ptr(logp_ref), clip_eps, kl_beta, adv_eps, _ptr(token_obj), result.data_ptr(), stream)
    if rc:
        raise TandemError(rc)
    r = result.cpu().numpy()
    return dict(loss=float(r[0]), clip_frac=float(r[1]), n_senior=int(r[2]), n_live=int(r[3]), result=result, token_obj=token_obj)


def tandem_test_uniforms(seed, seq_id, t, stream, n, out_dev):
    rc = lib().tandem_test_uniforms(seed, seq_id, t, stream, n, out_dev.data_ptr())
    if rc:
        raise TandemError(rc)


def tandem_test_nucleus(logits, temperature, top_p, u, token_out, keep_out, top_k=0):
    rc = lib().tandem_test_nucleus(logits.numel(), temperature, top_p, top_k, logits.data_ptr(), u.data_ptr(), token_out.data_ptr(), keep_out.data_ptr())
    if rc:
        raise TandemError(rc)


def tandem_test_philox(ctr, key):
    c = (C.c_uint32 * 4)(*ctr); k = (C.c_uint32 * 2)(*key); o = (C.c_uint32 * 4)()
    rc = lib().tandem_test_philox(c, k, o)
    if rc:
        raise TandemError(rc)
    return [int(x) for x in o]


def tandem_test_gemm(dtype, impl, A, W, out):
    rows, K = A.shape
    N = W.shape[0]
    rc = lib().tandem_test_gemm(dtype, impl, rows, N, K, A.data_ptr(), W.data_ptr(), out.data_ptr())
    if rc:
        raise TandemError(rc)


def tandem_test_gemm_time(rows, N, K, iters=50, ring_kb=0, splits=0, swiglu=0, pdl=0, pair=0):
    ms = C.c_float()
    rc = lib().tandem_test_gemm_time(rows, N, K, iters, ring_kb, splits, (1 if swiglu else 0) | (2 if pdl else 0) | (4 if pair else 0),
                                     C.byref(ms))
    if rc:
        raise TandemError(rc)
    return ms.value
