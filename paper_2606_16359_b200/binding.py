"""Thin ctypes binding of libfenc (include/fenc.h): argument marshalling only -- every step of the hot path
runs in the library's CUDA kernels.  PyTorch supplies device memory (allocator callbacks) and the stream.

There is no CPU fallback: importing works without a GPU (so that the symbol checks can run), but creating a
Context without a CUDA device raises."""
import ctypes as C
import os

import numpy as np

from . import build as _build

_HERE = os.path.dirname(os.path.abspath(__file__))
RELIN_KEY_ID = 1 << 40

STATUS = {0: "OK", 1: "INVALID_ARG", 2: "PARAMS", 3: "LAYOUT", 4: "NO_KEY", 5: "LEVEL", 6: "MISMATCH", 7: "OOM",
          8: "DEVICE", 9: "CUDA"}

ALLOC_FN = C.CFUNCTYPE(C.c_void_p, C.c_size_t, C.c_void_p)
FREE_FN = C.CFUNCTYPE(None, C.c_void_p, C.c_void_p)


class ParamsDesc(C.Structure):
    _fields_ = [("log2N", C.c_uint32), ("n_q", C.c_uint32), ("q_bits", C.c_uint32), ("n_p", C.c_uint32),
                ("p_bits", C.c_uint32), ("dnum", C.c_uint32), ("dlen_override", C.c_uint32),
                ("allow_noisy_ks", C.c_uint32), ("log2_scale", C.c_double),
                ("q_override", C.POINTER(C.c_uint64)), ("p_override", C.POINTER(C.c_uint64)),
                ("dev_alloc", ALLOC_FN), ("dev_free", FREE_FN), ("user", C.c_void_p),
                ("cuda_stream", C.c_void_p), ("device", C.c_int)]


class ConvDesc(C.Structure):
    _fields_ = [("BS", C.c_uint32), ("C_in", C.c_uint32), ("H", C.c_uint32), ("W", C.c_uint32), ("C_out", C.c_uint32),
                ("K", C.c_uint32), ("stride", C.c_uint32), ("pad", C.c_uint32), ("depthwise", C.c_int32),
                ("S", C.c_uint32), ("M", C.c_uint32), ("seg_v", C.c_uint32), ("B_cap", C.c_uint32), ("bsgs", C.c_uint32)]


class KeyMaterial(C.Structure):
    _fields_ = [("s", C.POINTER(C.c_int64)), ("n_keys", C.c_size_t), ("key_ids", C.POINTER(C.c_int64)),
                ("b", C.POINTER(C.POINTER(C.c_uint64))), ("a", C.POINTER(C.POINTER(C.c_uint64)))]


class FcDesc(C.Structure):
    _fields_ = [(k, C.c_uint32) for k in ("BS", "n_in", "n_out", "in_C", "in_H", "in_W", "in_M", "bsgs", "frag_in", "frag_out")]


class FcInfo(C.Structure):
    _fields_ = [(k, C.c_uint32) for k in ("B", "P", "BG", "n_in_ct", "n_out_ct", "n_rot", "n_pmult", "n_distinct_pt",
                                          "n_rot_keys", "bsgs")] + [("rot_steps", C.c_int32 * 512)]


class Layout(C.Structure):
    _fields_ = [(k, C.c_uint32) for k in ("S", "S_out", "M", "M_out", "m", "B", "ch", "cs", "G_in", "G_out", "BG",
                                          "H_out", "W_out", "n_in_ct", "n_out_ct", "n_inner_rot", "n_outer_rot",
                                          "n_pmult", "n_distinct_pt", "n_rot_keys", "ch_phys", "seg")] + \
               [("S_star_real", C.c_double), ("paper_rot_count", C.c_double), ("rot_steps", C.c_int32 * 512)]

    def steps(self):
        return [int(self.rot_steps[i]) for i in range(self.n_rot_keys)]


# every symbol include/fenc.h declares (checked by tests/test_abi.py against the header text)
SYMBOLS = ["fenc_params_init", "fenc_ctx_free", "fenc_last_error", "fenc_get_primes", "fenc_sync", "fenc_layout_plan",
           "fenc_keygen", "fenc_keys_free", "fenc_secret_export", "fenc_evk_export", "fenc_encode_fragment",
           "fenc_encode_slots", "fenc_pt_from_coeffs", "fenc_pt_coeffs", "fenc_pt_free", "fenc_encrypt",
           "fenc_decrypt_slots", "fenc_decrypt_decode", "fenc_ct_export", "fenc_ct_import", "fenc_ct_info",
           "fenc_ct_free", "fenc_rotate", "fenc_rescale", "fenc_add", "fenc_pmult_sum", "fenc_square_relin",
           "fenc_wts_keys", "fenc_conv_weights", "fenc_conv_weights_from_coeffs", "fenc_wts_free", "fenc_hconv",
           "fenc_compress", "fenc_ntt_rows", "fenc_launch_count", "fenc_device_bytes", "fenc_sum_groups",
           "fenc_profile_enable", "fenc_profile_kernels", "fenc_profile_name", "fenc_profile_read", "fenc_fc_plan",
           "fenc_fc_wts_keys", "fenc_fc_weights", "fenc_fc_weights_from_coeffs", "fenc_fc", "fenc_measure_alu_peak",
           "fenc_cmult_relin", "fenc_mul_scalar", "fenc_add_const", "fenc_ct_import_async", "fenc_ct_export_async",
           "fenc_export_wait", "fenc_set_hoisting", "fenc_rotate_hoisted", "fenc_square_sum_relin",
           "fenc_wts_factors", "fenc_wts_mask_slots", "fenc_conv_weights_factored", "fenc_conv_weights_factored_from_ints",
           "fenc_measure_smac_peak", "fenc_repack", "fenc_keys_import", "fenc_sum_pool", "fenc_square_sum_pool", "fenc_poly3",
           "fenc_rescale_static_prepare", "fenc_rescale_static", "fenc_fc_encode_input", "fenc_fc_decrypt_decode"]

_lib = None


def load_library(path=None):
    """dlopen libfenc.so (building it first if the sources are newer) and set the argument types."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    lib = C.CDLL(path or _build.build())
    vp, u64p, i64p, dp, i32p, u32p = C.c_void_p, C.POINTER(C.c_uint64), C.POINTER(C.c_int64), C.POINTER(C.c_double), \
        C.POINTER(C.c_int32), C.POINTER(C.c_uint32)
    vpp = C.POINTER(C.c_void_p)
    sig = {
        "fenc_params_init": [C.POINTER(ParamsDesc), vpp],
        "fenc_get_primes": [vp, u64p, u64p, u32p, u32p],
        "fenc_sync": [vp],
        "fenc_layout_plan": [vp, C.POINTER(ConvDesc), C.POINTER(Layout)],
        "fenc_keygen": [vp, C.c_uint64, i32p, C.c_size_t, C.c_int, vpp],
        "fenc_secret_export": [vp, vp, i64p],
        "fenc_evk_export": [vp, vp, C.c_int64, u64p, u64p],
        "fenc_encode_fragment": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), dp, C.c_uint32, C.c_uint32, C.c_uint32,
                                 C.c_uint32, C.c_uint32, C.c_double, vpp],
        "fenc_encode_slots": [vp, dp, dp, C.c_uint32, C.c_double, vpp],
        "fenc_pt_from_coeffs": [vp, i64p, C.c_uint32, C.c_double, vpp],
        "fenc_pt_coeffs": [vp, vp, i64p],
        "fenc_encrypt": [vp, vp, vp, C.c_uint64, vpp],
        "fenc_decrypt_slots": [vp, vp, vp, dp, dp],
        "fenc_decrypt_decode": [vp, vp, vp, C.POINTER(ConvDesc), C.POINTER(Layout), C.c_int, C.c_uint32, C.c_uint32,
                                C.c_uint32, C.c_uint32, dp],
        "fenc_ct_export": [vp, vp, u64p],
        "fenc_ct_import": [vp, u64p, C.c_uint32, C.c_double, vpp],
        "fenc_ct_import_async": [vp, u64p, C.c_uint32, C.c_double, vpp],
        "fenc_ct_export_async": [vp, vp, u64p],
        "fenc_export_wait": [vp],
        "fenc_set_hoisting": [vp, C.c_int],
        "fenc_square_sum_relin": [vp, vp, vpp, C.c_size_t, C.c_size_t, vpp],
        "fenc_rotate_hoisted": [vp, vp, vpp, C.c_size_t, i32p, C.c_size_t, vpp],
        "fenc_ct_info": [vp, vp, u32p, dp, vpp],
        "fenc_rotate": [vp, vp, vpp, i32p, C.c_size_t, vpp],
        "fenc_rescale": [vp, vpp, C.c_size_t, vpp],
        "fenc_add": [vp, vp, vp, vpp],
        "fenc_pmult_sum": [vp, vpp, vpp, C.c_size_t, vpp],
        "fenc_square_relin": [vp, vp, vpp, C.c_size_t, vpp],
        "fenc_sum_groups": [vp, vpp, C.c_size_t, C.c_size_t, vpp],
        "fenc_cmult_relin": [vp, vp, vpp, vpp, C.c_size_t, vpp],
        "fenc_mul_scalar": [vp, vpp, C.c_size_t, u64p, C.c_double, vpp],
        "fenc_add_const": [vp, vpp, C.c_size_t, u64p, vpp],
        "fenc_profile_enable": [vp, C.c_int],
        "fenc_measure_alu_peak": [vp, dp, dp],
        "fenc_measure_smac_peak": [vp, dp],
        "fenc_profile_read": [vp, dp, u64p, dp, dp, C.c_int],
        "fenc_wts_keys": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), u32p, C.c_size_t, C.POINTER(C.c_size_t)],
        "fenc_conv_weights": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), dp, C.c_uint32, C.c_double, vpp],
        "fenc_conv_weights_from_coeffs": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), i64p, C.c_size_t, C.c_uint32,
                                          C.c_double, vpp],
        "fenc_hconv": [vp, vp, C.POINTER(ConvDesc), C.POINTER(Layout), vp, vpp, C.c_size_t, C.c_int, vpp, C.c_size_t,
                       C.POINTER(C.c_size_t)],
        "fenc_wts_factors": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), u32p, C.c_size_t, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)],
        "fenc_wts_mask_slots": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), C.c_uint32, dp],
        "fenc_conv_weights_factored": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), dp, C.c_uint32, C.c_double, vpp],
        "fenc_conv_weights_factored_from_ints": [vp, C.POINTER(ConvDesc), C.POINTER(Layout), i64p, C.c_size_t, i64p, C.c_size_t,
                                                 C.c_uint32, C.c_double, C.c_double, vpp],
        "fenc_fc_plan": [vp, C.POINTER(FcDesc), C.POINTER(FcInfo)],
        "fenc_fc_wts_keys": [vp, C.POINTER(FcDesc), u32p, C.c_size_t, C.POINTER(C.c_size_t)],
        "fenc_fc_encode_input": [vp, C.POINTER(FcDesc), dp, C.c_uint32, C.c_uint32, C.c_uint32, C.c_double, vpp],
        "fenc_fc_decrypt_decode": [vp, vp, vp, C.POINTER(FcDesc), C.c_int, C.c_uint32, C.c_uint32, dp],
        "fenc_fc_weights": [vp, C.POINTER(FcDesc), dp, C.c_uint32, C.c_double, vpp],
        "fenc_fc_weights_from_coeffs": [vp, C.POINTER(FcDesc), i64p, C.c_size_t, C.c_uint32, C.c_double, vpp],
        "fenc_fc": [vp, vp, C.POINTER(FcDesc), vp, vpp, C.c_size_t, C.c_int, vpp, C.c_size_t, C.POINTER(C.c_size_t)],
        "fenc_compress": [vp, vp, vpp, C.c_size_t, vp, u32p, u32p, i32p, C.c_size_t, C.c_int, vpp, C.c_size_t],
        "fenc_ntt_rows": [vp, vp, i32p, C.c_size_t, C.c_int],
        "fenc_rescale_static_prepare": [vp, C.c_uint32],
        "fenc_rescale_static": [vp, vp, vp],
        "fenc_keys_import": [vp, C.POINTER(KeyMaterial), vpp],
        "fenc_sum_pool": [vp, vpp, C.c_size_t, C.c_uint32, vpp],
        "fenc_square_sum_pool": [vp, vp, vpp, C.c_size_t, C.c_uint32, vpp],
        "fenc_poly3": [vp, vp, vpp, C.c_size_t, u64p, u64p, u64p, C.c_double, vpp],
        "fenc_repack": [vp, vp, vpp, C.c_size_t, vpp, u32p, u32p, i32p, C.c_size_t, C.c_int, vpp, C.c_size_t],
    }
    for name, args in sig.items():
        f = getattr(lib, name)
        f.argtypes, f.restype = args, C.c_int
    for name in ("fenc_ctx_free", "fenc_keys_free", "fenc_pt_free", "fenc_ct_free", "fenc_wts_free"):
        getattr(lib, name).argtypes, getattr(lib, name).restype = [vp], None
    lib.fenc_last_error.argtypes, lib.fenc_last_error.restype = [vp], C.c_char_p
    lib.fenc_profile_kernels.argtypes, lib.fenc_profile_kernels.restype = [], C.c_int
    lib.fenc_profile_name.argtypes, lib.fenc_profile_name.restype = [C.c_int], C.c_char_p
    lib.fenc_launch_count.argtypes, lib.fenc_launch_count.restype = [vp, C.c_int], C.c_uint64
    lib.fenc_device_bytes.argtypes, lib.fenc_device_bytes.restype = [vp], C.c_uint64
    if path is None:
        _lib = lib
    return lib


class FencError(RuntimeError):
    pass


def _ptr(a, ty):
    return a.ctypes.data_as(C.POINTER(ty))


class _Handle:
    _free = None

    def __init__(self, ctx, h):
        self.ctx, self.h = ctx, h

    def free(self):
        if self.h:
            getattr(self.ctx.lib, self._free)(self.h)
            self.h = None

    def __del__(self):
        try:
            if self.ctx.h:
                self.free()
        except Exception:
            pass


class Keys(_Handle):
    _free = "fenc_keys_free"


class Plaintext(_Handle):
    _free = "fenc_pt_free"


class Weights(_Handle):
    _free = "fenc_wts_free"


class Ciphertext(_Handle):
    _free = "fenc_ct_free"

    def info(self):
        L, s, p = C.c_uint32(), C.c_double(), C.c_void_p()
        self.ctx._ck(self.ctx.lib.fenc_ct_info(self.ctx.h, self.h, C.byref(L), C.byref(s), C.byref(p)))
        return L.value, s.value, p.value

    @property
    def L(self):
        return self.info()[0]

    @property
    def scale(self):
        return self.info()[1]


class Context:
    """fenc_params_init + the calls of include/fenc.h with numpy marshalling."""

    def __init__(self, log2N, n_q, q_bits, n_p, p_bits, dnum=1, log2_scale=40, dlen=0, allow_noisy_ks=False,
                 q_override=None, p_override=None, device=0):
        import torch
        self.lib = load_library()
        self.h = None
        if not torch.cuda.is_available():
            raise FencError("libfenc needs a CUDA device (sm_100a); there is no CPU fallback")
        self._torch = torch
        self._blocks = {}
        dev = torch.device("cuda", device)

        def _alloc(nbytes, _user):
            try:
                t = torch.empty(int(nbytes), dtype=torch.uint8, device=dev)
            except Exception:
                return None
            self._blocks[t.data_ptr()] = t
            return t.data_ptr()

        def _free(p, _user):
            self._blocks.pop(p, None)

        self._alloc_cb, self._free_cb = ALLOC_FN(_alloc), FREE_FN(_free)
        d = ParamsDesc()
        d.log2N, d.n_q, d.q_bits, d.n_p, d.p_bits, d.dnum = log2N, n_q, q_bits, n_p, p_bits, dnum
        d.dlen_override, d.allow_noisy_ks, d.log2_scale = dlen, int(allow_noisy_ks), float(log2_scale)
        self._qo = np.asarray(q_override, dtype=np.uint64) if q_override is not None else None
        self._po = np.asarray(p_override, dtype=np.uint64) if p_override is not None else None
        d.q_override = _ptr(self._qo, C.c_uint64) if self._qo is not None else None
        d.p_override = _ptr(self._po, C.c_uint64) if self._po is not None else None
        d.dev_alloc, d.dev_free, d.user = self._alloc_cb, self._free_cb, None
        with torch.cuda.device(dev):
            d.cuda_stream = torch.cuda.current_stream().cuda_stream
        d.device = device
        h = C.c_void_p()
        st = self.lib.fenc_params_init(C.byref(d), C.byref(h))
        if st != 0:
            raise FencError("fenc_params_init: " + STATUS.get(st, str(st)))
        self.h = h
        self.log2N, self.N, self.n, self.n_q, self.n_p = log2N, 1 << log2N, 1 << (log2N - 1), n_q, n_p
        q = np.zeros(n_q, dtype=np.uint64)
        p = np.zeros(n_p, dtype=np.uint64)
        dl, bm = C.c_uint32(), C.c_uint32()
        self._ck(self.lib.fenc_get_primes(self.h, _ptr(q, C.c_uint64), _ptr(p, C.c_uint64), C.byref(dl), C.byref(bm)))
        self.q, self.p, self.dlen, self.beta_max = [int(x) for x in q], [int(x) for x in p], dl.value, bm.value

    def _ck(self, st):
        if st != 0:
            raise FencError("%s: %s" % (STATUS.get(st, str(st)), self.lib.fenc_last_error(self.h).decode()))

    def close(self):
        if self.h:
            self.lib.fenc_ctx_free(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sync(self):
        self._ck(self.lib.fenc_sync(self.h))

    def launch_count(self, reset=False):
        return int(self.lib.fenc_launch_count(self.h, int(reset)))

    def ct_bytes(self, ct):
        """device bytes of a ciphertext: uint64 [2][L][N]"""
        return 2 * ct.L * self.N * 8

    def device_bytes(self):
        return int(self.lib.fenc_device_bytes(self.h))

    # ---- planner
    def conv_desc(self, BS, C_in, H, W, C_out, K, stride=1, pad=0, depthwise=False, S=0, M=0, seg_v=0, B_cap=0, bsgs=1):
        """bsgs: baby steps over the channel diagonals (1 = plain, 0 = the library's choice, FENC_CONV_BSGS_AUTO)"""
        return ConvDesc(BS, C_in, H, W, C_out, K, stride, pad, int(depthwise), S, M, seg_v, B_cap, 0xFFFFFFFF if bsgs == 0 else bsgs)

    def layout_plan(self, conv):
        lay = Layout()
        self._ck(self.lib.fenc_layout_plan(self.h, C.byref(conv), C.byref(lay)))
        return lay

    # ---- keys
    def keygen(self, seed, rot_steps=(), want_relin=False):
        steps = np.asarray(list(rot_steps), dtype=np.int32)
        h = C.c_void_p()
        self._ck(self.lib.fenc_keygen(self.h, C.c_uint64(seed), _ptr(steps, C.c_int32), len(steps), int(want_relin), C.byref(h)))
        return Keys(self, h)

    def keys_import(self, s, evk):
        """host-generated key material uploaded verbatim: s int64[N] in {-1,0,1}; evk {key id: (b, a)} with b, a uint64
        [beta_max][n_q+n_p][N], coefficient domain (the format evk_export returns)"""
        s = np.ascontiguousarray(s, dtype=np.int64)
        ids = np.array(sorted(evk), dtype=np.int64)
        bs = [np.ascontiguousarray(evk[int(i)][0], dtype=np.uint64) for i in ids]
        as_ = [np.ascontiguousarray(evk[int(i)][1], dtype=np.uint64) for i in ids]
        PP = C.POINTER(C.c_uint64)
        mat = KeyMaterial(_ptr(s, C.c_int64), len(ids), _ptr(ids, C.c_int64) if len(ids) else None,
                          (PP * len(ids))(*[_ptr(x, C.c_uint64) for x in bs]), (PP * len(ids))(*[_ptr(x, C.c_uint64) for x in as_]))
        h = C.c_void_p()
        self._ck(self.lib.fenc_keys_import(self.h, C.byref(mat), C.byref(h)))
        return Keys(self, h)

    def secret_export(self, keys):
        s = np.zeros(self.N, dtype=np.int64)
        self._ck(self.lib.fenc_secret_export(self.h, keys.h, _ptr(s, C.c_int64)))
        return s

    def evk_export(self, keys, key_id):
        A = self.n_q + self.n_p
        b = np.zeros((self.beta_max, A, self.N), dtype=np.uint64)
        a = np.zeros_like(b)
        self._ck(self.lib.fenc_evk_export(self.h, keys.h, C.c_int64(key_id), _ptr(b, C.c_uint64), _ptr(a, C.c_uint64)))
        return b, a

    # ---- plaintexts
    def encode_fragment(self, conv, lay, x, u, v, g, bg, n_limbs, scale=0.0):
        x = np.ascontiguousarray(x, dtype=np.float64)
        assert x.shape == (conv.BS, conv.C_in, conv.H, conv.W)
        h = C.c_void_p()
        self._ck(self.lib.fenc_encode_fragment(self.h, C.byref(conv), C.byref(lay), _ptr(x, C.c_double), u, v, g, bg, n_limbs,
                                               float(scale), C.byref(h)))
        return Plaintext(self, h)

    def encode_slots(self, z, n_limbs, scale=0.0):
        z = np.asarray(z)
        re = np.ascontiguousarray(z.real, dtype=np.float64)
        im = np.ascontiguousarray(z.imag, dtype=np.float64) if np.iscomplexobj(z) else None
        assert re.shape == (self.n,)
        h = C.c_void_p()
        self._ck(self.lib.fenc_encode_slots(self.h, _ptr(re, C.c_double), _ptr(im, C.c_double) if im is not None else None,
                                            n_limbs, float(scale), C.byref(h)))
        return Plaintext(self, h)

    def pt_from_coeffs(self, coeffs, n_limbs, scale=0.0):
        c = np.ascontiguousarray(coeffs, dtype=np.int64)
        assert c.shape == (self.N,)
        h = C.c_void_p()
        self._ck(self.lib.fenc_pt_from_coeffs(self.h, _ptr(c, C.c_int64), n_limbs, float(scale), C.byref(h)))
        return Plaintext(self, h)

    def pt_coeffs(self, pt):
        c = np.zeros(self.N, dtype=np.int64)
        self._ck(self.lib.fenc_pt_coeffs(self.h, pt.h, _ptr(c, C.c_int64)))
        return c

    # ---- ciphertexts
    def encrypt(self, keys, pt, enc_seed):
        h = C.c_void_p()
        self._ck(self.lib.fenc_encrypt(self.h, keys.h, pt.h, C.c_uint64(enc_seed), C.byref(h)))
        return Ciphertext(self, h)

    def decrypt_slots(self, keys, ct):
        re = np.zeros(self.n, dtype=np.float64)
        im = np.zeros(self.n, dtype=np.float64)
        self._ck(self.lib.fenc_decrypt_slots(self.h, keys.h, ct.h, _ptr(re, C.c_double), _ptr(im, C.c_double)))
        return re + 1j * im

    def decrypt_decode(self, keys, ct, conv, lay, which, u, v, g, bg, y):
        assert y.dtype == np.float64 and y.flags["C_CONTIGUOUS"]
        self._ck(self.lib.fenc_decrypt_decode(self.h, keys.h, ct.h, C.byref(conv), C.byref(lay), which, u, v, g, bg,
                                              _ptr(y, C.c_double)))

    def ct_export(self, ct):
        L = ct.L
        out = np.zeros((2, L, self.N), dtype=np.uint64)
        self._ck(self.lib.fenc_ct_export(self.h, ct.h, _ptr(out, C.c_uint64)))
        return out

    def ct_import(self, limbs, scale=0.0):
        a = np.ascontiguousarray(limbs, dtype=np.uint64)
        assert a.ndim == 3 and a.shape[0] == 2 and a.shape[2] == self.N
        h = C.c_void_p()
        self._ck(self.lib.fenc_ct_import(self.h, _ptr(a, C.c_uint64), a.shape[1], float(scale), C.byref(h)))
        return Ciphertext(self, h)

    def ct_import_async(self, limbs, scale=0.0):
        """fenc_ct_import_async: `limbs` (a contiguous uint64 [2][L][N] array, page-locked for a real overlap) must stay
        alive and unchanged until the next synchronising call (sync, ct_export, decrypt)."""
        a = limbs
        assert a.dtype == np.uint64 and a.flags.c_contiguous and a.ndim == 3 and a.shape[0] == 2 and a.shape[2] == self.N
        h = C.c_void_p()
        self._ck(self.lib.fenc_ct_import_async(self.h, _ptr(a, C.c_uint64), a.shape[1], float(scale), C.byref(h)))
        return Ciphertext(self, h)

    def ct_export_async(self, ct, out):
        """fenc_ct_export_async into `out` (contiguous uint64 [2][L][N], page-locked for a real overlap); valid after
        export_wait()."""
        assert out.dtype == np.uint64 and out.flags.c_contiguous and out.shape == (2, ct.L, self.N)
        self._ck(self.lib.fenc_ct_export_async(self.h, ct.h, _ptr(out, C.c_uint64)))

    def set_hoisting(self, on=True):
        """inner rotations of hconv / fc in the hoisted form (R2.7b); compare with the oracle's hoist=True runs"""
        self._ck(self.lib.fenc_set_hoisting(self.h, int(bool(on))))

    def export_wait(self):
        self._ck(self.lib.fenc_export_wait(self.h))

    def rotate_hoisted(self, keys, cts, steps):
        """every ciphertext by every amount, one decomposition per ciphertext (R2.7b) -> list [ct][step]"""
        st = np.asarray(list(steps), dtype=np.int32)
        n, m = len(cts), len(st)
        out = (C.c_void_p * (n * m))()
        self._ck(self.lib.fenc_rotate_hoisted(self.h, keys.h, self._harr(cts), n, _ptr(st, C.c_int32), m, out))
        return [[Ciphertext(self, C.c_void_p(out[i * m + s])) for s in range(m)] for i in range(n)]

    def _harr(self, handles):
        return (C.c_void_p * len(handles))(*[x.h.value for x in handles])

    # ---- primitives
    def rotate(self, keys, cts, steps):
        n = len(cts)
        st = np.asarray(list(steps), dtype=np.int32)
        assert st.shape == (n,)
        out = (C.c_void_p * n)()
        self._ck(self.lib.fenc_rotate(self.h, keys.h, self._harr(cts), _ptr(st, C.c_int32), n, out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n)]

    def rescale(self, cts):
        n = len(cts)
        out = (C.c_void_p * n)()
        self._ck(self.lib.fenc_rescale(self.h, self._harr(cts), n, out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n)]

    def rescale_static_prepare(self, L):
        """set-up of rescale_static for level L (may allocate)"""
        self._ck(self.lib.fenc_rescale_static_prepare(self.h, int(L)))

    def rescale_static(self, ct, out):
        """out := rescale(ct) with no device allocation: `out` is an existing ciphertext at L-1 limbs (fenc.h)"""
        self._ck(self.lib.fenc_rescale_static(self.h, ct.h, out.h))
        return out

    def add(self, a, b):
        h = C.c_void_p()
        self._ck(self.lib.fenc_add(self.h, a.h, b.h, C.byref(h)))
        return Ciphertext(self, h)

    def pmult_sum(self, cts, pts):
        h = C.c_void_p()
        self._ck(self.lib.fenc_pmult_sum(self.h, self._harr(cts), self._harr(pts), len(cts), C.byref(h)))
        return Ciphertext(self, h)

    def square_relin(self, keys, cts):
        single = isinstance(cts, Ciphertext)
        lst = [cts] if single else list(cts)
        out = (C.c_void_p * len(lst))()
        self._ck(self.lib.fenc_square_relin(self.h, keys.h, self._harr(lst), len(lst), out))
        res = [Ciphertext(self, C.c_void_p(out[i])) for i in range(len(lst))]
        return res[0] if single else res

    def square_sum_relin(self, keys, cts, group):
        """consecutive groups of `group` ciphertexts -> sum of their squares with one relinearisation each (R2.12c)"""
        lst = list(cts)
        assert group >= 1 and len(lst) % group == 0
        n = len(lst) // group
        out = (C.c_void_p * n)()
        self._ck(self.lib.fenc_square_sum_relin(self.h, keys.h, self._harr(lst), n, group, out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n)]

    def cmult_relin(self, keys, a, b):
        out = (C.c_void_p * len(a))()
        self._ck(self.lib.fenc_cmult_relin(self.h, keys.h, self._harr(a), self._harr(b), len(a), out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(len(a))]

    def _residues(self, k, L):
        return np.asarray([int(k) % self.q[t] for t in range(L)], dtype=np.uint64)

    def mul_scalar(self, cts, k, scale_factor):
        """every limb times the (Python) integer k; the scale is multiplied by scale_factor."""
        r = self._residues(k, cts[0].L)
        out = (C.c_void_p * len(cts))()
        self._ck(self.lib.fenc_mul_scalar(self.h, self._harr(cts), len(cts), _ptr(r, C.c_uint64), float(scale_factor), out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(len(cts))]

    def add_const(self, cts, k):
        """the (Python) integer k added to coefficient 0 of c0."""
        r = self._residues(k, cts[0].L)
        out = (C.c_void_p * len(cts))()
        self._ck(self.lib.fenc_add_const(self.h, self._harr(cts), len(cts), _ptr(r, C.c_uint64), out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(len(cts))]

    def sum_groups(self, cts, group):
        n = len(cts) // group
        assert n * group == len(cts)
        out = (C.c_void_p * n)()
        self._ck(self.lib.fenc_sum_groups(self.h, self._harr(cts), group, n, out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n)]

    def sum_pool(self, cts, S):
        out = (C.c_void_p * (len(cts) // 4))()
        self._ck(self.lib.fenc_sum_pool(self.h, self._harr(cts), len(cts), int(S), out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(len(cts) // 4)]

    def square_sum_pool(self, keys, cts, S):
        out = (C.c_void_p * (len(cts) // 4))()
        self._ck(self.lib.fenc_square_sum_pool(self.h, keys.h, self._harr(cts), len(cts), int(S), out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(len(cts) // 4)]

    def poly3(self, keys, cts, k3, k1, k0, scale_sq):
        """the three exactly rounded integers of the degree-3 activation (fenc.h fenc_poly3), as Python ints"""
        L = cts[0].L
        r3, r1, r0 = self._residues(k3, L), self._residues(k1, L), self._residues(k0, L - 2)
        out = (C.c_void_p * len(cts))()
        self._ck(self.lib.fenc_poly3(self.h, keys.h, self._harr(cts), len(cts), _ptr(r3, C.c_uint64), _ptr(r1, C.c_uint64),
                                     _ptr(r0, C.c_uint64), float(scale_sq), out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(len(cts))]

    def measure_alu_peak(self):
        a, b = C.c_double(), C.c_double()
        self._ck(self.lib.fenc_measure_alu_peak(self.h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def measure_smac_peak(self):
        v = C.c_double()
        self._ck(self.lib.fenc_measure_smac_peak(self.h, C.byref(v)))
        return v.value

    def profile_enable(self, on=True):
        self._ck(self.lib.fenc_profile_enable(self.h, int(on)))

    def profile_read(self, reset=True):
        """{kernel class: (ms, launches, algorithmic bytes, modular butterflies)} accumulated since the last reset."""
        k = self.lib.fenc_profile_kernels()
        ms, cnt, by, op = np.zeros(k), np.zeros(k, dtype=np.uint64), np.zeros(k), np.zeros(k)
        self._ck(self.lib.fenc_profile_read(self.h, _ptr(ms, C.c_double), _ptr(cnt, C.c_uint64), _ptr(by, C.c_double),
                                            _ptr(op, C.c_double), int(reset)))
        return {self.lib.fenc_profile_name(i).decode(): (float(ms[i]), int(cnt[i]), float(by[i]), float(op[i]))
                for i in range(k) if cnt[i]}

    # ---- HConv
    def wts_keys(self, conv, lay):
        n = C.c_size_t()
        self._ck(self.lib.fenc_wts_keys(self.h, C.byref(conv), C.byref(lay), None, 0, C.byref(n)))
        k = np.zeros((n.value, 7), dtype=np.uint32)
        self._ck(self.lib.fenc_wts_keys(self.h, C.byref(conv), C.byref(lay), _ptr(k, C.c_uint32), n.value, C.byref(n)))
        return k

    def conv_weights(self, conv, lay, w, n_limbs, scale=0.0):
        w = np.ascontiguousarray(w, dtype=np.float64)
        h = C.c_void_p()
        self._ck(self.lib.fenc_conv_weights(self.h, C.byref(conv), C.byref(lay), _ptr(w, C.c_double), n_limbs, float(scale), C.byref(h)))
        return Weights(self, h)

    def conv_weights_from_coeffs(self, conv, lay, coeffs, n_limbs, scale=0.0):
        c = np.ascontiguousarray(coeffs, dtype=np.int64)
        assert c.ndim == 2 and c.shape[1] == self.N
        h = C.c_void_p()
        self._ck(self.lib.fenc_conv_weights_from_coeffs(self.h, C.byref(conv), C.byref(lay), _ptr(c, C.c_int64), c.shape[0],
                                                        n_limbs, float(scale), C.byref(h)))
        return Weights(self, h)

    # ---- factored weights (R2.9c)
    def wts_factors(self, conv, lay):
        """(mask id of every weight in wts_keys order, number of distinct masks)"""
        n, nm = C.c_size_t(), C.c_size_t()
        self._ck(self.lib.fenc_wts_factors(self.h, C.byref(conv), C.byref(lay), None, 0, C.byref(n), C.byref(nm)))
        m = np.zeros(n.value, dtype=np.uint32)
        self._ck(self.lib.fenc_wts_factors(self.h, C.byref(conv), C.byref(lay), _ptr(m, C.c_uint32), n.value, C.byref(n), C.byref(nm)))
        return m, nm.value

    def wts_mask_slots(self, conv, lay, mask_id):
        v = np.zeros(self.n, dtype=np.float64)
        self._ck(self.lib.fenc_wts_mask_slots(self.h, C.byref(conv), C.byref(lay), int(mask_id), _ptr(v, C.c_double)))
        return v

    def conv_weights_factored(self, conv, lay, w, n_limbs, scale=0.0):
        w = np.ascontiguousarray(w, dtype=np.float64)
        h = C.c_void_p()
        self._ck(self.lib.fenc_conv_weights_factored(self.h, C.byref(conv), C.byref(lay), _ptr(w, C.c_double), n_limbs, float(scale), C.byref(h)))
        return Weights(self, h)

    def conv_weights_factored_from_ints(self, conv, lay, k, mask_coeffs, n_limbs, E1, E2):
        k = np.ascontiguousarray(k, dtype=np.int64)
        mc = np.ascontiguousarray(mask_coeffs, dtype=np.int64)
        assert mc.ndim == 2 and mc.shape[1] == self.N
        h = C.c_void_p()
        self._ck(self.lib.fenc_conv_weights_factored_from_ints(self.h, C.byref(conv), C.byref(lay), _ptr(k, C.c_int64), k.shape[0],
                                                               _ptr(mc, C.c_int64), mc.shape[0], n_limbs, float(E1), float(E2), C.byref(h)))
        return Weights(self, h)

    def hconv(self, keys, conv, lay, wts, cts, do_rescale=True):
        cap = int(lay.n_out_ct)
        out = (C.c_void_p * cap)()
        n = C.c_size_t()
        self._ck(self.lib.fenc_hconv(self.h, keys.h, C.byref(conv), C.byref(lay), wts.h, self._harr(cts), len(cts),
                                     int(do_rescale), out, cap, C.byref(n)))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n.value)]

    # ---- FC by plain diagonals
    def fc_desc(self, BS, n_in, n_out, in_C=0, in_H=0, in_W=0, in_M=1, bsgs=1, frag_in=0, frag_out=0):
        """bsgs: baby-step count g (1 = plain diagonals, 0 = the library's choice, FENC_FC_BSGS_AUTO);
        frag_in / frag_out: sub-block sizes S / S' of fragment-encoded embeddings (include/fenc.h, R2.13)"""
        return FcDesc(BS, n_in, n_out, in_C, in_H, in_W, in_M, 0xFFFFFFFF if bsgs == 0 else bsgs, frag_in, frag_out)

    def fc_plan(self, fc):
        info = FcInfo()
        self._ck(self.lib.fenc_fc_plan(self.h, C.byref(fc), C.byref(info)))
        d = {k: int(getattr(info, k)) for k, _ in FcInfo._fields_ if k != "rot_steps"}
        d["rot_steps"] = [int(info.rot_steps[i]) for i in range(info.n_rot_keys)]
        return d

    def fc_encode_input(self, fc, x, c, bg, n_limbs, scale=0.0):
        x = np.ascontiguousarray(x, dtype=np.float64)
        assert x.shape == (fc.BS, fc.n_in)
        h = C.c_void_p()
        self._ck(self.lib.fenc_fc_encode_input(self.h, C.byref(fc), _ptr(x, C.c_double), c, bg, n_limbs, float(scale), C.byref(h)))
        return Plaintext(self, h)

    def fc_decrypt_decode(self, keys, ct, fc, side, c, bg, y):
        assert y.dtype == np.float64 and y.flags["C_CONTIGUOUS"] and y.shape == (fc.BS, fc.n_out if side else fc.n_in)
        self._ck(self.lib.fenc_fc_decrypt_decode(self.h, keys.h, ct.h, C.byref(fc), side, c, bg, _ptr(y, C.c_double)))

    def fc_wts_keys(self, fc):
        n = C.c_size_t()
        self._ck(self.lib.fenc_fc_wts_keys(self.h, C.byref(fc), None, 0, C.byref(n)))
        k = np.zeros((n.value, 3), dtype=np.uint32)
        self._ck(self.lib.fenc_fc_wts_keys(self.h, C.byref(fc), _ptr(k, C.c_uint32), n.value, C.byref(n)))
        return k

    def fc_weights(self, fc, w, n_limbs, scale=0.0):
        w = np.ascontiguousarray(w, dtype=np.float64)
        assert w.shape == (fc.n_out, fc.n_in)
        h = C.c_void_p()
        self._ck(self.lib.fenc_fc_weights(self.h, C.byref(fc), _ptr(w, C.c_double), n_limbs, float(scale), C.byref(h)))
        return Weights(self, h)

    def fc_weights_from_coeffs(self, fc, coeffs, n_limbs, scale=0.0):
        c = np.ascontiguousarray(coeffs, dtype=np.int64)
        assert c.ndim == 2 and c.shape[1] == self.N
        h = C.c_void_p()
        self._ck(self.lib.fenc_fc_weights_from_coeffs(self.h, C.byref(fc), _ptr(c, C.c_int64), c.shape[0], n_limbs, float(scale),
                                                      C.byref(h)))
        return Weights(self, h)

    def fc(self, keys, fc, wts, cts, do_rescale=True):
        cap = self.fc_plan(fc)["n_out_ct"]
        out = (C.c_void_p * cap)()
        n = C.c_size_t()
        self._ck(self.lib.fenc_fc(self.h, keys.h, C.byref(fc), wts.h, self._harr(cts), len(cts), int(do_rescale), out, cap, C.byref(n)))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n.value)]

    def compress(self, keys, cts, terms, n_out, mask=None, do_rescale=False):
        """terms: list of (out index, source index, rotation amount)."""
        to = np.asarray([t[0] for t in terms], dtype=np.uint32)
        ts = np.asarray([t[1] for t in terms], dtype=np.uint32)
        tr = np.asarray([t[2] for t in terms], dtype=np.int32)
        out = (C.c_void_p * n_out)()
        self._ck(self.lib.fenc_compress(self.h, keys.h, self._harr(cts), len(cts), mask.h if mask is not None else None,
                                        _ptr(to, C.c_uint32), _ptr(ts, C.c_uint32), _ptr(tr, C.c_int32), len(terms),
                                        int(do_rescale), out, n_out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n_out)]

    # ---- raw NTT on a torch tensor of uint64 rows (viewed as int64 by torch)
    def repack(self, keys, cts, terms, n_out, do_rescale=True):
        """terms: list of (output index, source index, rotation amount, mask Plaintext) -- rot-mask-add (R2.11c)"""
        to = np.array([t[0] for t in terms], dtype=np.uint32)
        ts = np.array([t[1] for t in terms], dtype=np.uint32)
        tr = np.array([t[2] for t in terms], dtype=np.int32)
        out = (C.c_void_p * n_out)()
        self._ck(self.lib.fenc_repack(self.h, keys.h, self._harr(cts), len(cts), self._harr([t[3] for t in terms]),
                                      _ptr(to, C.c_uint32), _ptr(ts, C.c_uint32), _ptr(tr, C.c_int32), len(terms), int(do_rescale), out, n_out))
        return [Ciphertext(self, C.c_void_p(out[i])) for i in range(n_out)]

    def ntt_rows(self, tensor, mod_idx, inverse=False):
        m = np.asarray(list(mod_idx), dtype=np.int32)
        assert tensor.is_cuda and tensor.is_contiguous() and tensor.numel() == len(m) * self.N
        self._ck(self.lib.fenc_ntt_rows(self.h, C.c_void_p(tensor.data_ptr()), _ptr(m, C.c_int32), len(m), int(inverse)))
