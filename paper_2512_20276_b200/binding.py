"""Thin ctypes binding of include/af.h — argument marshalling only; every step of the path runs in the CUDA kernels.

PyTorch is used for device memory (tensor.data_ptr()) and streams only.  Loading fails loudly when the CUDA
library has not been built (python -m paper_2512_20276_b200.build, or __graft_entry__.build()).
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libaf_b200.so")

AF_OK, AF_ERR_ARG, AF_ERR_SEGMENT, AF_ERR_POSITION = 0, -1, -2, -3
AF_ERR_CAPACITY, AF_ERR_WORKSPACE, AF_ERR_CUDA, AF_ERR_UNSUPPORTED = -4, -5, -6, -7
ERR_NAMES = {0: "AF_OK", -1: "AF_ERR_ARG", -2: "AF_ERR_SEGMENT", -3: "AF_ERR_POSITION", -4: "AF_ERR_CAPACITY",
             -5: "AF_ERR_WORKSPACE", -6: "AF_ERR_CUDA", -7: "AF_ERR_UNSUPPORTED"}


class AfError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERR_NAMES.get(code, code)}: {msg}")
        self.code = code
        self.name = ERR_NAMES.get(code, str(code))


class af_model_cfg(C.Structure):
    _fields_ = [("d_model", C.c_int32), ("n_layers", C.c_int32), ("n_heads", C.c_int32), ("head_dim", C.c_int32),
                ("ffn", C.c_int32), ("vocab", C.c_int32), ("rms_eps", C.c_float), ("rope_theta", C.c_float)]


class af_ring_cfg(C.Structure):
    _fields_ = [("n_regions", C.c_int32), ("capacity", C.c_int32)]


class af_segment(C.Structure):
    _fields_ = [("req_id", C.c_int32), ("phase", C.c_int32), ("start_pos", C.c_int32), ("len", C.c_int32)]


class af_layer_weights(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("wq", "wk", "wv", "wo", "w_gate", "w_up", "w_down", "g_attn", "g_mlp")]


class af_layer_scales(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("sq", "sk", "sv", "so", "s_gate", "s_up", "s_down")]


class af_weights(C.Structure):
    _fields_ = [("cfg", af_model_cfg), ("layers", C.POINTER(af_layer_weights)), ("g_final", C.c_void_p),
                ("w_lm", C.c_void_p), ("weight_format", C.c_int32), ("scales", C.POINTER(af_layer_scales))]


EXPORTS = ["af_prepare_gate_up_fp8", "af_ring_set_window", "af_loop_create", "af_loop_buffers", "af_loop_step", "af_loop_steps_done", "af_loop_destroy",
           "af_argmax_rows", "af_argmax_rows_static", "af_embed_rows", "af_convert_bf16_to_fp16", "af_gate_up_rows", "af_prepare_gate_up", "af_ring_bytes", "af_workspace_bytes", "af_ring_create", "af_ring_reset_slot", "af_packed_forward",
           "af_logits_rows", "af_ring_destroy", "af_ring_get_state", "af_debug_row_map", "af_debug_set_len",
           "af_debug_launch_count", "af_debug_gemm", "af_debug_gemm_schedule", "af_debug_profile", "af_debug_attention", "af_debug_profile_read", "af_debug_trace", "af_debug_trace_read", "af_last_error"]

PROFILE_CLASSES = ["gemm_qkv", "gemm_o", "gemm_gateup", "gemm_down", "gemm_lm", "attention", "rope_append",
                   "rmsnorm", "chain", "other"]

_lib = None


def load_library():
    """dlopen the C-ABI library and declare its prototypes.  Raises if the library is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build the CUDA library first "
                           "(python -m paper_2512_20276_b200.build). There is no CPU fallback.")
    L = C.CDLL(LIB_PATH)
    vp, i32, sz = C.c_void_p, C.c_int32, C.c_size_t
    L.af_ring_bytes.restype = sz
    L.af_ring_bytes.argtypes = [C.POINTER(af_model_cfg), C.POINTER(af_ring_cfg)]
    L.af_workspace_bytes.restype = sz
    L.af_workspace_bytes.argtypes = [C.POINTER(af_model_cfg), i32, i32]
    L.af_convert_bf16_to_fp16.argtypes = [vp, vp, sz, vp]
    L.af_convert_bf16_to_fp16.restype = C.c_int
    L.af_argmax_rows.argtypes = [vp, C.c_int32, C.c_int32, vp, vp]
    L.af_argmax_rows.restype = C.c_int
    L.af_argmax_rows_static.argtypes = [vp, C.c_int32, C.c_int32, vp, vp]
    L.af_argmax_rows_static.restype = C.c_int
    L.af_embed_rows.argtypes = [vp, C.c_int32, C.c_int32, vp, C.c_int32, vp, vp]
    L.af_embed_rows.restype = C.c_int
    L.af_gate_up_rows.argtypes = [C.c_int32]
    L.af_gate_up_rows.restype = C.c_size_t
    L.af_prepare_gate_up.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, vp]
    L.af_prepare_gate_up.restype = C.c_int
    L.af_prepare_gate_up_fp8.argtypes = [vp, vp, vp, C.c_int32, C.c_int32, vp]
    L.af_prepare_gate_up_fp8.restype = C.c_int
    L.af_ring_create.argtypes = [C.POINTER(af_model_cfg), C.POINTER(af_ring_cfg), vp, sz, C.POINTER(vp)]
    L.af_ring_reset_slot.argtypes = [vp, i32, i32]
    L.af_ring_set_window.argtypes = [vp, i32, i32]
    L.af_ring_set_window.restype = C.c_int
    L.af_packed_forward.argtypes = [C.POINTER(af_weights), vp, C.POINTER(af_segment), i32, vp, vp, vp, sz, vp]
    L.af_logits_rows.argtypes = [C.POINTER(af_weights), vp, C.POINTER(i32), i32, vp, vp, sz, vp]
    L.af_ring_destroy.argtypes = [vp]
    L.af_ring_get_state.argtypes = [vp, i32, C.POINTER(i32), C.POINTER(i32)]
    L.af_debug_row_map.argtypes = [vp, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32), i32]
    L.af_debug_set_len.argtypes = [vp, i32, i32]
    L.af_debug_launch_count.restype = C.c_int64
    L.af_debug_launch_count.argtypes = []
    L.af_debug_gemm.argtypes = [vp, vp, vp, i32, i32, i32, vp, sz, vp]
    L.af_debug_profile.argtypes = [C.c_int]
    L.af_debug_profile.restype = C.c_int
    L.af_debug_profile_read.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_int64), i32]
    L.af_debug_profile_read.restype = C.c_int
    L.af_loop_create.argtypes = [C.POINTER(af_weights), vp, vp, i32, i32, vp, sz, C.POINTER(vp)]
    L.af_loop_buffers.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp), C.POINTER(vp)]
    L.af_loop_step.argtypes = [vp, i32, vp]
    L.af_loop_steps_done.argtypes = [vp]
    L.af_loop_destroy.argtypes = [vp]
    for n in ("af_loop_create", "af_loop_buffers", "af_loop_step", "af_loop_steps_done", "af_loop_destroy"):
        getattr(L, n).restype = C.c_int
    L.af_last_error.restype = C.c_char_p
    L.af_last_error.argtypes = []
    for n in ("af_ring_create", "af_ring_reset_slot", "af_packed_forward", "af_logits_rows", "af_ring_destroy",
              "af_ring_get_state", "af_debug_row_map", "af_debug_set_len", "af_debug_gemm"):
        getattr(L, n).restype = C.c_int
    _lib = L
    return L


def _check(rc):
    if rc != 0:
        raise AfError(rc, load_library().af_last_error().decode())


def _cfg_struct(cfg) -> af_model_cfg:
    return af_model_cfg(cfg.d_model, cfg.n_layers, cfg.n_heads, cfg.head_dim, cfg.ffn, cfg.vocab,
                        cfg.rms_eps, cfg.rope_theta)


def _stream_ptr(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Weights:
    """Device copies of the bf16 weights + the af_weights struct pointing at them.  With prepared=True (default) the
    projection matrices are rewritten once, on the device, as fp16 by af_convert_bf16_to_fp16 and gate | up are
    interleaved by af_prepare_gate_up (AF_WEIGHTS_FP16_GU: the same values, no per-tile conversion in the GEMM, one
    TMA box per gate/up tile); prepared="fp16" converts only (AF_WEIGHTS_FP16); prepared=False keeps them bf16
    (AF_WEIGHTS_BF16)."""

    def __init__(self, cfg, host_weights: dict, device="cuda", prepared=True):
        self.cfg = cfg
        self.prepared = prepared
        self.tensors = []          # keep alive
        self._layers = (af_layer_weights * cfg.n_layers)()
        for l, L in enumerate(host_weights["layers"]):
            for name, _ in af_layer_weights._fields_:
                if prepared is True and name in ("w_gate", "w_up"):
                    continue
                t = self._prep(L[name].to(torch.bfloat16).contiguous().to(device), name.startswith("w"))
                self.tensors.append(t)
                setattr(self._layers[l], name, t.data_ptr())
            if prepared is True:
                gate = L["w_gate"].to(torch.bfloat16).contiguous().to(device)
                up = L["w_up"].to(torch.bfloat16).contiguous().to(device)
                lib = load_library()
                gu = torch.empty(lib.af_gate_up_rows(cfg.ffn), cfg.d_model, dtype=torch.float16, device=device)
                _check(lib.af_prepare_gate_up(gate.data_ptr(), up.data_ptr(), gu.data_ptr(), cfg.ffn, cfg.d_model, _stream_ptr()))
                torch.cuda.synchronize()
                self.tensors.append(gu)
                self._layers[l].w_gate = gu.data_ptr()
                self._layers[l].w_up = gu.data_ptr()
        self.g_final = host_weights["g_final"].to(torch.bfloat16).contiguous().to(device)
        self.w_lm = self._prep(host_weights["w_lm"].to(torch.bfloat16).contiguous().to(device), True)
        torch.cuda.synchronize()
        self.struct = af_weights(_cfg_struct(cfg), self._layers, self.g_final.data_ptr(), self.w_lm.data_ptr(),
                                 2 if prepared is True else (1 if prepared else 0), None)

    def _prep(self, t: torch.Tensor, is_matrix: bool) -> torch.Tensor:
        if not (self.prepared and is_matrix):
            return t
        out = torch.empty(t.shape, dtype=torch.float16, device=t.device)
        _check(load_library().af_convert_bf16_to_fp16(t.data_ptr(), out.data_ptr(), t.numel(), _stream_ptr()))
        return out


class WeightsFP8:
    """f4: AF_WEIGHTS_FP8.  `quantized` is inputs.quantize_weights_fp8(host_weights): per projection matrix (E4M3 codes
    uint8 [out, in], fp32 scale [out]).  The codes go to the device as they are (gate | up interleaved by
    af_prepare_gate_up_fp8, a byte permutation), the scales as fp32 vectors; gains stay bf16 and the LM head a prepared
    fp16 matrix."""

    _SCALE_OF = {"wq": "sq", "wk": "sk", "wv": "sv", "wo": "so", "w_gate": "s_gate", "w_up": "s_up", "w_down": "s_down"}

    def __init__(self, cfg, quantized: dict, device="cuda"):
        lib = load_library()
        self.cfg = cfg
        self.tensors = []
        self._layers = (af_layer_weights * cfg.n_layers)()
        self._scales = (af_layer_scales * cfg.n_layers)()
        for l, L in enumerate(quantized["layers"]):
            for name, sname in self._SCALE_OF.items():
                codes, scale = L[name]
                sc = scale.to(torch.float32).contiguous().to(device)
                self.tensors.append(sc)
                setattr(self._scales[l], sname, sc.data_ptr())
                if name in ("w_gate", "w_up"):
                    continue
                cd = codes.contiguous().to(device)
                self.tensors.append(cd)
                setattr(self._layers[l], name, cd.data_ptr())
            gate, up = L["w_gate"][0].contiguous().to(device), L["w_up"][0].contiguous().to(device)
            gu = torch.empty(lib.af_gate_up_rows(cfg.ffn), cfg.d_model, dtype=torch.uint8, device=device)
            _check(lib.af_prepare_gate_up_fp8(gate.data_ptr(), up.data_ptr(), gu.data_ptr(), cfg.ffn, cfg.d_model, _stream_ptr()))
            torch.cuda.synchronize()
            self.tensors.append(gu)
            self._layers[l].w_gate = gu.data_ptr()
            self._layers[l].w_up = gu.data_ptr()
            for name in ("g_attn", "g_mlp"):
                t = L[name].to(torch.bfloat16).contiguous().to(device)
                self.tensors.append(t)
                setattr(self._layers[l], name, t.data_ptr())
        self.g_final = quantized["g_final"].to(torch.bfloat16).contiguous().to(device)
        lm = quantized["w_lm"].to(torch.bfloat16).contiguous().to(device)
        self.w_lm = torch.empty(lm.shape, dtype=torch.float16, device=device)
        _check(lib.af_convert_bf16_to_fp16(lm.data_ptr(), self.w_lm.data_ptr(), lm.numel(), _stream_ptr()))
        torch.cuda.synchronize()
        self.struct = af_weights(_cfg_struct(cfg), self._layers, self.g_final.data_ptr(), self.w_lm.data_ptr(), 3, self._scales)


class Ring:
    """af_ring_create / af_ring_reset_slot / af_packed_forward / af_logits_rows / af_ring_destroy."""

    def __init__(self, cfg, n_regions: int, capacity: int, max_rows: int, device="cuda"):
        L = load_library()
        self.cfg, self.R, self.Cap = cfg, n_regions, capacity
        self._c = _cfg_struct(cfg)
        self._r = af_ring_cfg(n_regions, capacity)
        nbytes = L.af_ring_bytes(C.byref(self._c), C.byref(self._r))
        self.kv_mem = torch.empty(nbytes, dtype=torch.uint8, device=device)
        self.max_rows = max_rows
        self.ws_bytes = L.af_workspace_bytes(C.byref(self._c), max_rows, 64)
        self.workspace = torch.empty(self.ws_bytes, dtype=torch.uint8, device=device)
        h = C.c_void_p()
        _check(L.af_ring_create(C.byref(self._c), C.byref(self._r), self.kv_mem.data_ptr(), nbytes, C.byref(h)))
        self.handle = h

    def kv_view(self) -> torch.Tensor:
        """The ring as fp16 [n_layers, 2, R, H, C, hd] (layout documented in include/af.h)."""
        c = self.cfg
        return self.kv_mem.view(torch.float16).view(c.n_layers, 2, self.R, c.n_heads, self.Cap, c.head_dim)

    def reset_slot(self, req_id: int, new_base: int = -1):
        _check(load_library().af_ring_reset_slot(self.handle, req_id, new_base))

    def set_window(self, window: int, max_pos: int = 0):
        _check(load_library().af_ring_set_window(self.handle, window, max_pos))

    def get_state(self, req_id: int):
        b, n = C.c_int32(), C.c_int32()
        _check(load_library().af_ring_get_state(self.handle, req_id, C.byref(b), C.byref(n)))
        return b.value, n.value

    def set_len(self, req_id: int, n: int):
        _check(load_library().af_debug_set_len(self.handle, req_id, n))

    def packed_forward(self, weights: Weights, packed_embeds: torch.Tensor, segs, hidden_out: torch.Tensor = None,
                       stream=None) -> torch.Tensor:
        T = sum(s[3] for s in segs)
        arr = (af_segment * max(1, len(segs)))(*[af_segment(*s) for s in segs])
        if hidden_out is None:
            hidden_out = torch.empty(T, self.cfg.d_model, dtype=torch.float32, device=packed_embeds.device)
        _check(load_library().af_packed_forward(C.byref(weights.struct), packed_embeds.data_ptr(), arr, len(segs),
                                                self.handle, hidden_out.data_ptr(), self.workspace.data_ptr(),
                                                self.ws_bytes, _stream_ptr(stream)))
        return hidden_out

    def logits_rows(self, weights: Weights, hidden: torch.Tensor, rows, logits_out: torch.Tensor = None, stream=None):
        n = len(rows)
        arr = (C.c_int32 * max(1, n))(*rows)
        if logits_out is None:
            logits_out = torch.empty(n, self.cfg.vocab, dtype=torch.float32, device=hidden.device)
        _check(load_library().af_logits_rows(C.byref(weights.struct), hidden.data_ptr(), arr, n, logits_out.data_ptr(),
                                             self.workspace.data_ptr(), self.ws_bytes, _stream_ptr(stream)))
        return logits_out

    def row_map(self, n: int):
        a, b, c = (C.c_int32 * max(1, n))(), (C.c_int32 * max(1, n))(), (C.c_int32 * max(1, n))()
        _check(load_library().af_debug_row_map(self.handle, a, b, c, n))
        return list(a)[:n], list(b)[:n], list(c)[:n]

    def destroy(self):
        if self.handle is not None:
            load_library().af_ring_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def debug_gemm(a: torch.Tensor, w: torch.Tensor) -> torch.Tensor:
    """out[n_tok, n_out] fp32 = a[n_tok, k] (fp16 activations) @ w[n_out, k]^T (bf16 weights), tcgen05 GEMM kernel."""
    L = load_library()
    assert a.dtype == torch.float16 and w.dtype == torch.bfloat16
    n_tok, k = a.shape
    n_out = w.shape[0]
    out = torch.empty(n_tok, n_out, dtype=torch.float32, device=a.device)
    ws = torch.empty(160 * 512 * 128 * 4, dtype=torch.uint8, device=a.device)
    _check(L.af_debug_gemm(a.data_ptr(), w.data_ptr(), out.data_ptr(), n_tok, n_out, k, ws.data_ptr(), ws.numel(),
                           _stream_ptr()))
    return out


def launch_count() -> int:
    return int(load_library().af_debug_launch_count())


def profile(enable: bool):
    _check(load_library().af_debug_profile(1 if enable else 0))


def attention_mode(mode: int):
    """af_debug_attention: 0 = automatic (units for decode-only steps), 1 = attention_kernel (mma.sync) always, 2 = the units
    of attention_umma.cuh wherever they apply."""
    L = load_library()
    L.af_debug_attention.argtypes, L.af_debug_attention.restype = [C.c_int], C.c_int
    _check(L.af_debug_attention(int(mode)))


def profile_read() -> dict:
    """{class: (sum_ms, launches)} since the last read (CUDA events on the launching stream)."""
    n = len(PROFILE_CLASSES)
    ms, cnt = (C.c_double * n)(), (C.c_int64 * n)()
    _check(load_library().af_debug_profile_read(ms, cnt, n))
    return {k: (ms[i], cnt[i]) for i, k in enumerate(PROFILE_CLASSES)}


def chain_trace(enable: bool):
    """af_debug_trace: switch the layer-chain kernel's per-phase %globaltimer stamps on / off (synchronises)."""
    L = load_library()
    L.af_debug_trace.argtypes, L.af_debug_trace.restype = [C.c_int], C.c_int
    _check(L.af_debug_trace(int(enable)))   # 2: the attention_umma_kernel launches' stamps instead of the chain's


def chain_trace_read():
    """(stamps int64 [16][160][18], meta int32 [16][2] = (phases, grid), launches recorded) of the last 16 chain launches."""
    import numpy as np
    L = load_library()
    L.af_debug_trace_read.argtypes, L.af_debug_trace_read.restype = [C.c_void_p, C.c_void_p], C.c_int
    st, meta = np.zeros((16, 160, 18), dtype=np.int64), np.zeros((16, 2), dtype=np.int32)
    n = L.af_debug_trace_read(st.ctypes.data, meta.ctypes.data)
    if n < 0:
        _check(n)
    return st, meta, n


def argmax_rows(logits: torch.Tensor) -> torch.Tensor:
    """af_argmax_rows: int32 [n] = lowest index of the maximum of every row of fp32 logits [n, V] (device)."""
    assert logits.is_cuda and logits.dtype == torch.float32 and logits.dim() == 2 and logits.is_contiguous()
    out = torch.empty(logits.shape[0], dtype=torch.int32, device=logits.device)
    _check(load_library().af_argmax_rows(logits.data_ptr(), logits.shape[0], logits.shape[1], out.data_ptr(), _stream_ptr()))
    return out


def argmax_rows_static(logits: torch.Tensor, out: torch.Tensor) -> torch.Tensor:
    """af_argmax_rows_static: af_argmax_rows without any allocation in the library (static device scratch, at most
    AF_ARGMAX_STATIC_MAX_ROWS = 256 rows); `out` is the caller's int32 [n] device tensor."""
    assert logits.is_cuda and logits.dtype == torch.float32 and logits.dim() == 2 and logits.is_contiguous()
    assert out.is_cuda and out.dtype == torch.int32 and out.is_contiguous() and out.numel() >= logits.shape[0]
    _check(load_library().af_argmax_rows_static(logits.data_ptr(), logits.shape[0], logits.shape[1], out.data_ptr(), _stream_ptr()))
    return out


def embed_rows(table: torch.Tensor, tokens: torch.Tensor, out: torch.Tensor = None) -> torch.Tensor:
    """af_embed_rows: out[i] = table[tokens[i]] for a bf16 table [V, D] and int32 tokens [n] (all device)."""
    assert table.is_cuda and table.dtype == torch.bfloat16 and table.is_contiguous() and tokens.dtype == torch.int32
    if out is None:
        out = torch.empty(tokens.shape[0], table.shape[1], dtype=torch.bfloat16, device=table.device)
    _check(load_library().af_embed_rows(table.data_ptr(), table.shape[0], table.shape[1], tokens.data_ptr(),
                                        tokens.shape[0], out.data_ptr(), _stream_ptr()))
    return out


def _wrap_device(ptr: int, dtype, shape, device):
    """A torch view of library-owned device memory (no copy, no ownership)."""
    iface = {"shape": tuple(shape), "typestr": {torch.float32: "<f4", torch.int32: "<i4", torch.int16: "<i2"}[dtype],
             "data": (ptr, False), "version": 2}
    holder = type("_DevMem", (), {"__cuda_array_interface__": iface})()
    return torch.as_tensor(holder, device=device)


class Loop:
    """af_loop_create / af_loop_buffers / af_loop_step / af_loop_destroy: Algorithm 1's pipeline with device-side state."""

    def __init__(self, weights: "Weights", ring: "Ring", embed_table: torch.Tensor, prefill_len: int, chunk_k: int):
        L = load_library()
        assert embed_table.dtype == torch.bfloat16 and embed_table.is_contiguous()
        self.weights, self.ring, self.table = weights, ring, embed_table        # keep the caller-owned memory alive
        self.L_P, self.K = prefill_len, chunk_k
        h = C.c_void_p()
        _check(L.af_loop_create(C.byref(weights.struct), ring.handle, embed_table.data_ptr(), prefill_len, chunk_k,
                                ring.workspace.data_ptr(), ring.ws_bytes, C.byref(h)))
        self.handle = h
        p = [C.c_void_p() for _ in range(5)]
        _check(L.af_loop_buffers(h, *[C.byref(x) for x in p]))
        cfg, dev = ring.cfg, embed_table.device
        T = prefill_len + chunk_k - 1
        # bf16 has no __cuda_array_interface__ typestr: view the embeddings as int16 and reinterpret
        self.prefill_embeds = _wrap_device(p[0].value, torch.int16,
                                           (prefill_len, cfg.d_model), dev).view(torch.bfloat16)
        self.hidden = _wrap_device(p[1].value, torch.float32, (T, cfg.d_model), dev)
        self.logits = _wrap_device(p[2].value, torch.float32, (chunk_k, cfg.vocab), dev)
        self.tokens = _wrap_device(p[3].value, torch.int32, (chunk_k,), dev)
        self.frame = _wrap_device(p[4].value, torch.int32, (1 + chunk_k,), dev)

    def step(self, use_graph: bool = True, stream=None):
        _check(load_library().af_loop_step(self.handle, 1 if use_graph else 0, _stream_ptr(stream)))

    @property
    def steps_done(self) -> int:
        return load_library().af_loop_steps_done(self.handle)

    def destroy(self):
        if self.handle is not None:
            load_library().af_loop_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
