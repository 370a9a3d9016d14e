"""libcrypto EVP_MAC("SIPHASH") through ctypes — an implementation independent of oracle/ and of
the CUDA path, used only to pin the oracle (SURVEY.md §8(c) pin (iv))."""
import ctypes as C
import ctypes.util


class _OsslParam(C.Structure):
    _fields_ = [("key", C.c_char_p), ("data_type", C.c_uint), ("data", C.c_void_p),
                ("data_size", C.c_size_t), ("return_size", C.c_size_t)]


_OSSL_PARAM_UNSIGNED_INTEGER = 2


class OpenSSLSipHash:
    def __init__(self):
        name = ctypes.util.find_library("crypto") or "libcrypto.so.3"
        L = C.CDLL(name)
        L.EVP_MAC_fetch.restype = C.c_void_p
        L.EVP_MAC_fetch.argtypes = [C.c_void_p, C.c_char_p, C.c_char_p]
        L.EVP_MAC_CTX_new.restype = C.c_void_p
        L.EVP_MAC_CTX_new.argtypes = [C.c_void_p]
        L.EVP_MAC_init.restype = C.c_int
        L.EVP_MAC_init.argtypes = [C.c_void_p, C.c_char_p, C.c_size_t, C.c_void_p]
        L.EVP_MAC_update.restype = C.c_int
        L.EVP_MAC_update.argtypes = [C.c_void_p, C.c_char_p, C.c_size_t]
        L.EVP_MAC_final.restype = C.c_int
        L.EVP_MAC_final.argtypes = [C.c_void_p, C.c_char_p, C.POINTER(C.c_size_t), C.c_size_t]
        self.L = L
        self.mac = L.EVP_MAC_fetch(None, b"SIPHASH", None)
        if not self.mac:
            raise RuntimeError("libcrypto has no SIPHASH MAC")
        self.ctx = L.EVP_MAC_CTX_new(self.mac)
        self._size = C.c_uint(8)
        self._params = (_OsslParam * 2)()
        self._params[0] = _OsslParam(b"size", _OSSL_PARAM_UNSIGNED_INTEGER,
                                     C.cast(C.pointer(self._size), C.c_void_p), C.sizeof(self._size), 0)
        self._params[1] = _OsslParam(None, 0, None, 0, 0)
        self._out = C.create_string_buffer(16)
        self._outl = C.c_size_t(0)

    def __call__(self, key: bytes, msg: bytes) -> int:
        L = self.L
        assert len(key) == 16
        assert L.EVP_MAC_init(self.ctx, key, 16, C.cast(self._params, C.c_void_p)) == 1
        assert L.EVP_MAC_update(self.ctx, msg, len(msg)) == 1
        assert L.EVP_MAC_final(self.ctx, self._out, C.byref(self._outl), 16) == 1
        assert self._outl.value == 8
        return int.from_bytes(self._out.raw[:8], "little")


def get():
    try:
        return OpenSSLSipHash()
    except Exception:
        return None
