"""TEST INFRASTRUCTURE: lets the `-m gpu` test files run on a box without a GPU, as a dry run --
`HOUGH_GPU_TESTS_ON_EMULATOR=1 python -m pytest tests/test_parity_gpu.py tests/test_parity_next_gpu.py -m gpu` --
through the package's real Python binding and the product's real host code, every kernel launch executed by the SIMT
emulator (tests/simt_emu/host.py).  It finds mistakes in the test files themselves and in the binding before GPU
minutes are spent on them, and repeats the parity checks at reduced event counts.  It proves nothing about the device
code and is never on by default: a normal run skips every gpu-marked test on a box without a GPU (tests/conftest.py).

What is faked: torch tensors stay on the CPU (`.cuda()` is an aligned copy, `device="cuda"` and `pin_memory()` are identities), streams are
numbered objects, synchronisation is a no-op, the package's library handle is the host-emulated library, and the input
generator shrinks batches of more than 250 events to HOUGH_EMU_MAX_EVENTS (default 8)."""
import contextlib
import itertools
import os


class FakeStream:
    _ids = itertools.count(1)

    def __init__(self, *a, **k):
        self.cuda_stream = next(FakeStream._ids)

    def synchronize(self):
        pass

    def wait_stream(self, other):
        pass

    def wait_event(self, ev):
        pass


class FakeEvent:
    def __init__(self, *a, **k):
        pass

    def record(self, stream=None):
        pass

    def synchronize(self):
        pass

    def elapsed_time(self, other):
        return 1.0


def install():
    import torch

    import paper_2607_04067_b200 as hb
    import stcf_inputs as si

    from . import host

    lib = host.load(race=os.environ.get("HOUGH_EMU_RACE") == "1")
    hb._lib = lib                                            # load_library() returns it from now on
    real_check = hb._marshal_check
    hb._marshal_check = lambda cuda, *a, **k: real_check(False, *a, **k)      # every check but "is a CUDA tensor"
    hb._is_device_tensor = lambda t: isinstance(t, torch.Tensor)
    hb._stream_handle = lambda stream: None if stream is None else __import__("ctypes").c_void_p(stream.cuda_stream)

    current = FakeStream()
    current.cuda_stream = 0
    torch.cuda.is_available = lambda: True
    torch.cuda.device_count = lambda: 1
    torch.cuda.synchronize = lambda *a, **k: None
    torch.cuda.Stream = FakeStream
    torch.cuda.Event = FakeEvent
    torch.cuda.current_stream = lambda *a, **k: current
    torch.cuda.stream = lambda s: contextlib.nullcontext()
    torch.cuda.empty_cache = lambda: None
    def to_device(self, *a, **k):          # a copy in its own 256-byte aligned allocation, as cudaMalloc gives
        nbytes = self.numel() * self.element_size()
        buf = torch.empty(nbytes + 256, dtype=torch.uint8)
        start = (-buf.data_ptr()) % 256
        out = buf[start:start + nbytes].view(self.dtype).reshape(self.shape)
        out.copy_(self)
        return out
    torch.Tensor.cuda = to_device
    torch.Tensor.pin_memory = lambda self, *a, **k: self

    def on_cpu(fn):
        def wrapped(*a, **k):
            dev = k.get("device")
            if dev is not None and "cuda" in str(dev):
                k["device"] = "cpu"
            return fn(*a, **k)
        return wrapped
    for name in ("empty", "zeros", "full", "ones", "tensor"):
        setattr(torch, name, on_cpu(getattr(torch, name)))

    cap = int(os.environ.get("HOUGH_EMU_MAX_EVENTS", "8"))
    real_generate = si.generate

    def generate(w, n_events=None, *a, **k):      # only the big batches shrink: small requests keep the count the test relies on
        n = w.n_events if n_events is None else n_events
        return real_generate(w, cap if n > 250 else n, *a, **k)
    si.generate = generate
    return lib
