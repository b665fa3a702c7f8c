"""ctypes binding of include/dex.h — argument marshalling only; every step of the path runs in
the CUDA kernels behind the C ABI.  PyTorch is used for device memory and the stream."""
import ctypes as C
import os

import numpy as np

DEX_OK, DEX_EINVAL, DEX_ECAPACITY, DEX_ESTATE, DEX_ECUDA = 0, -1, -2, -3, -4
DEX_MAX_DEPTHS = 8
DEX_STEP_AUTOCOLLAPSE = 1
DEX_TAP_HIDDEN, DEX_TAP_LOGITS, DEX_TAP_B, DEX_TAP_FSM, DEX_TAP_ROUND_TIMES, DEX_TAP_REF_BLOCKS = 1, 2, 3, 4, 5, 6

_HERE = os.path.dirname(os.path.abspath(__file__))
lib_path = os.path.join(_HERE, "libdex_b200.so")


class DexError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"dex error {code}: {msg}")
        self.code = code


class DexConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("n_layers", "d_model", "n_heads", "n_kv_heads", "head_dim", "d_ffn", "vocab")] + \
               [("rms_eps", C.c_float), ("rope_theta", C.c_float)] + \
               [(n, C.c_int32) for n in ("max_seqs", "max_ctx", "page_size", "decs", "eos_id", "debug_taps",
                                         "act_planes", "use_graph", "round_kernel", "sample")] + \
               [("temperature", C.c_float), ("sample_seed", C.c_int32), ("adapter_dim", C.c_int32), ("lookahead", C.c_int32)]


class DexWeights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("embed", "lm_head", "wqkv", "wo", "wgu", "wdn",
                                          "norm_attn", "norm_ffn", "norm_final",
                                          "ad_w1", "ad_w2", "ad_b1", "ad_b2", "ad_norm", "ad_alpha")]


class DexStepResult(C.Structure):
    _fields_ = [("active", C.c_int32), ("committed", C.c_int32), ("token", C.c_int32), ("match_k", C.c_int32),
                ("q_before", C.c_int32), ("q_after", C.c_int32), ("exit_rows", C.c_int32),
                ("critical_layers", C.c_int32), ("layer_evals", C.c_int64),
                ("rows_per_stage", C.c_int32 * DEX_MAX_DEPTHS), ("anchor_tokens", C.c_int32 * DEX_MAX_DEPTHS),
                ("ref_top1", C.c_float), ("ref_top2", C.c_float), ("n_tokens", C.c_int32), ("done", C.c_int32),
                ("branch_mask", C.c_int32), ("reserved", C.c_int32)]


_SIGNATURES = {
    "dex_workspace_bytes": (C.c_int32, [C.POINTER(DexConfig), C.POINTER(C.c_int32), C.c_int32, C.POINTER(C.c_size_t)]),
    "dex_init": (C.c_int32, [C.POINTER(C.c_void_p), C.POINTER(DexConfig), C.POINTER(DexWeights), C.POINTER(C.c_int32),
                             C.c_int32, C.c_void_p, C.c_size_t, C.c_void_p]),
    "dex_prefill": (C.c_int32, [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.c_int32]),
    "dex_step": (C.c_int32, [C.c_void_p, C.c_uint32, C.POINTER(DexStepResult)]),
    "dex_collapse": (C.c_int32, [C.c_void_p, C.c_int32, C.c_int32, C.c_int32]),
    "dex_rewind": (C.c_int32, [C.c_void_p, C.c_int32, C.c_int32]),
    "dex_get_tokens": (C.c_int32, [C.c_void_p, C.c_int32, C.POINTER(C.c_int32), C.c_int32, C.POINTER(C.c_int32)]),
    "dex_debug_read": (C.c_int32, [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_size_t]),
    "dex_debug_gemm": (C.c_int32, [C.c_void_p, C.c_int32, C.c_int32, C.POINTER(C.c_float), C.c_int32, C.POINTER(C.c_float)]),
    "dex_debug_phase_us": (C.c_int32, [C.c_void_p, C.POINTER(C.c_float)]),
    "dex_profile": (C.c_int32, [C.c_void_p, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_double)]),
    "dex_gemm_noalloc": (C.c_int32, [C.c_void_p, C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_void_p, C.c_void_p]),
    "dex_destroy": (C.c_int32, [C.c_void_p]),
    "dex_last_error": (C.c_char_p, [C.c_void_p]),
}
exported_symbols = tuple(_SIGNATURES)

_lib = None


def lib():
    """Load libdex_b200.so.  Fails loudly when the CUDA extension has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(lib_path):
            raise ImportError(f"{lib_path} is missing: build it with `python -m paper_2606_29223_b200.build` "
                              "(there is no CPU fallback)")
        _lib = C.CDLL(lib_path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(_lib, name)
            fn.restype, fn.argtypes = res, args
    return _lib


def dex_last_error(ctx=None):
    return lib().dex_last_error(ctx).decode()


def _check(rc, ctx=None):
    if rc != DEX_OK:
        raise DexError(rc, dex_last_error(ctx))


def _i32arr(v):
    a = np.ascontiguousarray(v, dtype=np.int32)
    return a, a.ctypes.data_as(C.POINTER(C.c_int32))


def dex_workspace_bytes(cfg, depths):
    d, dp = _i32arr(depths)
    out = C.c_size_t(0)
    _check(lib().dex_workspace_bytes(C.byref(cfg), dp, len(d), C.byref(out)))
    return out.value


def dex_init(cfg, weights, depths, workspace_ptr, workspace_bytes, stream_ptr):
    d, dp = _i32arr(depths)
    ctx = C.c_void_p()
    _check(lib().dex_init(C.byref(ctx), C.byref(cfg), C.byref(weights), dp, len(d), workspace_ptr, workspace_bytes,
                          stream_ptr))
    return ctx


def dex_prefill(ctx, seq, prompt):
    p, pp = _i32arr(prompt)
    _check(lib().dex_prefill(ctx, seq, pp, len(p)), ctx)


def dex_step(ctx, flags, results):
    _check(lib().dex_step(ctx, flags, results), ctx)


def dex_collapse(ctx, seq, branch_k, token):
    _check(lib().dex_collapse(ctx, seq, branch_k, token), ctx)


def dex_rewind(ctx, seq, n):
    _check(lib().dex_rewind(ctx, seq, n), ctx)


def dex_get_tokens(ctx, seq, cap):
    out = np.zeros(cap, dtype=np.int32)
    n = C.c_int32(0)
    _check(lib().dex_get_tokens(ctx, seq, out.ctypes.data_as(C.POINTER(C.c_int32)), cap, C.byref(n)), ctx)
    return out[:min(cap, n.value)]


def dex_debug_read(ctx, what, seq, a, out_array):
    _check(lib().dex_debug_read(ctx, what, seq, a, out_array.ctypes.data_as(C.c_void_p), out_array.nbytes), ctx)
    return out_array


def dex_debug_gemm(ctx, which, layer, x, out_dim):
    x = np.ascontiguousarray(x, dtype=np.float32)
    y = np.zeros((x.shape[0], out_dim), dtype=np.float32)
    _check(lib().dex_debug_gemm(ctx, which, layer, x.ctypes.data_as(C.POINTER(C.c_float)), x.shape[0],
                                y.ctypes.data_as(C.POINTER(C.c_float))), ctx)
    return y


def dex_debug_phase_us(ctx):
    out = np.zeros(8, dtype=np.float32)
    _check(lib().dex_debug_phase_us(ctx, out.ctypes.data_as(C.POINTER(C.c_float))), ctx)
    return out


def dex_profile(ctx, on):
    ph, ct = np.zeros(8, dtype=np.float64), np.zeros(8, dtype=np.float64)
    _check(lib().dex_profile(ctx, on, ph.ctypes.data_as(C.POINTER(C.c_double)), ct.ctypes.data_as(C.POINTER(C.c_double))), ctx)
    return ph, ct


def dex_gemm_noalloc(w_ptr, x_ptr, rows, out_dim, k_dim, act_planes, y_ptr, stream_ptr):
    """y = x . W^T through the allocation-free entry point; all pointers are DEVICE addresses (ints)."""
    _check(lib().dex_gemm_noalloc(w_ptr, x_ptr, rows, out_dim, k_dim, act_planes, y_ptr, stream_ptr))


def dex_destroy(ctx):
    _check(lib().dex_destroy(ctx))


class Dex:
    """Convenience owner of the device memory a context borrows (weights, workspace, stream)."""

    def __init__(self, shape, weights, depths, max_seqs=1, max_ctx=1024, page_size=128, decs=1, eos_id=-1,
                 debug_taps=0, act_planes=2, use_graph=1, round_kernel=1, sample=0, temperature=1.0, sample_seed=0,
                 adapters=None, lookahead=0, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_29223_b200 needs a CUDA device (no CPU fallback)")
        self.torch = torch
        self.device = torch.device(device)
        self.shape, self.depths = shape, tuple(int(d) for d in depths)
        adapter_dim = 0
        if adapters is not None:            # dex_synth.make_adapters layout: one adapter per non-final depth
            if adapters["w1"].shape[0] != len(self.depths) - 1:
                raise ValueError("need one inducing adapter per non-final depth (N - 1)")
            adapter_dim = int(adapters["w1"].shape[1])
        self.cfg = DexConfig(shape.n_layers, shape.d_model, shape.n_heads, shape.n_kv_heads, shape.head_dim,
                             shape.d_ffn, shape.vocab, shape.rms_eps, shape.rope_theta, max_seqs, max_ctx, page_size,
                             decs, eos_id, debug_taps, act_planes, use_graph, round_kernel, sample, temperature,
                             sample_seed, adapter_dim, lookahead)
        with torch.cuda.device(self.device):
            self.w = {}
            for k, v in weights.items():
                dt = torch.float32 if k.startswith("norm") else torch.bfloat16
                self.w[k] = v.to(device=self.device, dtype=dt).contiguous()
            ptrs = [self.w[k].data_ptr() for k in ("embed", "lm_head", "wqkv", "wo", "wgu", "wdn",
                                                   "norm_attn", "norm_ffn", "norm_final")]
            if adapters is not None:
                for k in ("w1", "w2", "b1", "b2", "norm", "alpha"):
                    dt = torch.bfloat16 if k in ("w1", "w2") else torch.float32
                    self.w["ad_" + k] = adapters[k].to(device=self.device, dtype=dt).contiguous()
                    ptrs.append(self.w["ad_" + k].data_ptr())
            else:
                ptrs += [None] * 6
            self.wstruct = DexWeights(*ptrs)
            self.ws_bytes = dex_workspace_bytes(self.cfg, self.depths)
            self.workspace = torch.empty(self.ws_bytes + 1024, dtype=torch.uint8, device=self.device)
            ptr = (self.workspace.data_ptr() + 1023) // 1024 * 1024
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            torch.cuda.synchronize(self.device)
            self.ctx = dex_init(self.cfg, self.wstruct, self.depths, ptr, self.ws_bytes, self.stream.cuda_stream)
        self.results = (DexStepResult * max_seqs)()
        self.max_seqs = max_seqs

    def prefill(self, seq, prompt):
        dex_prefill(self.ctx, seq, prompt)

    def step(self, flags=DEX_STEP_AUTOCOLLAPSE):
        dex_step(self.ctx, flags, self.results)
        return self.results

    def collapse(self, seq, branch_k, token):
        dex_collapse(self.ctx, seq, branch_k, token)

    def rewind(self, seq, n):
        dex_rewind(self.ctx, seq, n)

    def tokens(self, seq=0, cap=None):
        return dex_get_tokens(self.ctx, seq, cap or (self.cfg.max_ctx + 1))

    def generate(self, n_new, seq=0, flags=DEX_STEP_AUTOCOLLAPSE):
        """Run rounds until `n_new` tokens are committed for `seq`; returns (tokens, per-round records)."""
        out, recs = [], []
        while len(out) < n_new:
            r = self.step(flags)[seq]
            recs.append(dict(q=r.q_before, committed=r.committed, token=r.token, match_k=r.match_k,
                             layer_evals=r.layer_evals, critical_layers=r.critical_layers,
                             rows_per_stage=list(r.rows_per_stage), exit_rows=r.exit_rows,
                             ref_top1=r.ref_top1, ref_top2=r.ref_top2, branch_mask=r.branch_mask))
            if r.committed:
                out.append(r.token)
            if r.done or not r.active:
                break
        return np.array(out, dtype=np.int64), recs

    def tap_hidden(self, node, seq=0):
        level = int(np.floor(np.log2(node + 1)))
        o = node + 1 - (1 << level)
        m = level if o == 0 else (o & -o).bit_length() - 1
        lo = 0 if m == 0 else self.depths[m - 1]
        out = np.zeros((self.depths[m] - lo, self.shape.d_model), dtype=np.float32)
        return dex_debug_read(self.ctx, DEX_TAP_HIDDEN, seq, node, out)

    def tap_logits(self, seq=0):
        return dex_debug_read(self.ctx, DEX_TAP_LOGITS, seq, 0, np.zeros(self.shape.vocab, dtype=np.float32))

    def tap_ref_blocks(self, seq=0):
        """(top-1, top-2) of every 32-id vocabulary block as reduced by the fused exit epilogue: [n_blocks, 2]."""
        n = 4 * ((self.shape.vocab + 127) // 128)
        return dex_debug_read(self.ctx, DEX_TAP_REF_BLOCKS, seq, 0, np.zeros((n, 2), dtype=np.float32))

    def tap_B(self, seq=0):
        return dex_debug_read(self.ctx, DEX_TAP_B, seq, 0, np.zeros((1 << len(self.depths)) - 1, dtype=np.int32))

    def tap_fsm(self, seq=0):
        return dex_debug_read(self.ctx, DEX_TAP_FSM, seq, 0, np.zeros(4, dtype=np.int32))

    def tap_round_times(self):
        n = 20 * max(b - a for a, b in zip((0,) + self.depths[:-1], self.depths)) + 68
        return dex_debug_read(self.ctx, DEX_TAP_ROUND_TIMES, 0, 0, np.zeros(n, dtype=np.uint64))

    def gemm(self, which, layer, x):
        outs = (self.shape.qkv_out, self.shape.d_model, 2 * self.shape.d_ffn, self.shape.d_model)
        return dex_debug_gemm(self.ctx, which, layer, x, outs[which])

    def profile(self, on):
        return dex_profile(self.ctx, on)

    def phase_us(self):
        return dex_debug_phase_us(self.ctx)

    def close(self):
        if getattr(self, "ctx", None) is not None:
            dex_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
