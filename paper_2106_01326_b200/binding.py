"""ctypes binding of include/vox.h.  Marshalling only; torch supplies device memory and streams."""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# VOX_LIB selects another build of the same library (tests: the checked build libvox_checked.so)
_LIB_PATH = os.environ.get("VOX_LIB") or os.path.join(_HERE, "libvox.so")
_lib = None

# every symbol include/vox.h declares
EXPORTS = [
    "vox_create", "vox_destroy", "vox_set_tile", "vox_set_variant", "vox_tets", "vox_grid_words",
    "vox_workspace_bytes", "vox_workspace_fixed_bytes", "vox_plan", "vox_run", "vox_status",
    "vox_validate", "vox_host_arena_bytes", "vox_run_host", "vox_timing_enable", "vox_timing_read",
    "vox_probe_int32", "vox_strerror", "vox_last_error",
    "vox_pipe_create", "vox_pipe_destroy", "vox_pipe_set_variant", "vox_pipe_set_tile", "vox_pipe_arena_bytes",
    "vox_pipe_bind", "vox_pipe_submit", "vox_pipe_wait", "vox_pipe_last_error",
    "vox_tile_shape", "vox_run_sparse", "vox_sparse_status", "vox_pipe_submit_sparse", "vox_pipe_tile_shape",
    "vox_pipe_reserve_pairs", "vox_occupancy", "vox_lattice", "vox_pipe_submit_lattice", "vox_kernel_launches",
    "vox_debug_check_status", "vox_run_noalloc", "vox_path", "vox_debug_selftest",
]


NOALLOC_SCRATCH_BYTES = 4 << 20  # include/vox.h VOX_NOALLOC_SCRATCH_BYTES


class VoxError(RuntimeError):
    def __init__(self, code, where, detail=""):
        self.code = code
        super().__init__(f"{where}: {_strerror(code)} ({code}){' -- ' + detail if detail else ''}")


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen libvox.so (built by paper_2106_01326_b200.build).  No fallback."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: run `python -m paper_2106_01326_b200.build` "
            "(or __graft_entry__.build()).  There is no CPU fallback."
        )
    lib = ctypes.CDLL(_LIB_PATH)
    vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_int64, ctypes.c_size_t
    sig = {
        "vox_create": (i32, [ctypes.POINTER(vp), i32, i32, i32, i32, i32, i32, i32]),
        "vox_destroy": (None, [vp]),
        "vox_set_tile": (i32, [vp, i32, i32]),
        "vox_set_variant": (i32, [vp, i32]),
        "vox_tets": (i32, [vp, vp, i64, vp, i64, vp]),
        "vox_grid_words": (sz, [vp]),
        "vox_workspace_bytes": (sz, [vp]),
        "vox_workspace_fixed_bytes": (sz, [vp]),
        "vox_plan": (i32, [vp, vp, vp, sz, ctypes.POINTER(i64)]),
        "vox_run": (i32, [vp, vp, vp, sz, vp]),
        "vox_status": (i32, [vp, vp, vp, ctypes.POINTER(i64)]),
        "vox_validate": (i32, [vp, vp, vp, sz]),
        "vox_host_arena_bytes": (sz, [vp, i64, i64]),
        "vox_run_host": (i32, [vp, vp, vp, i64, vp, i64, vp, vp, sz, vp]),
        "vox_timing_enable": (i32, [vp, i32]),
        "vox_timing_read": (i32, [vp, i32, ctypes.POINTER(ctypes.c_float)]),
        "vox_probe_int32": (i32, [vp, i32, i32, i32, vp, ctypes.POINTER(ctypes.c_double)]),
        "vox_strerror": (ctypes.c_char_p, [i32]),
        "vox_last_error": (ctypes.c_char_p, [vp]),
        "vox_pipe_create": (i32, [ctypes.POINTER(vp), i32, i32, i32, i32, i32, i32, i32, i32, i64, i64]),
        "vox_pipe_destroy": (None, [vp]),
        "vox_pipe_set_variant": (i32, [vp, i32]),
        "vox_pipe_set_tile": (i32, [vp, i32, i32]),
        "vox_pipe_arena_bytes": (sz, [vp]),
        "vox_pipe_bind": (i32, [vp, vp, sz]),
        "vox_pipe_submit": (i32, [vp, vp, i64, vp, i64, vp, vp, ctypes.POINTER(i64)]),
        "vox_pipe_wait": (i32, [vp, i64, ctypes.POINTER(i64)]),
        "vox_pipe_last_error": (ctypes.c_char_p, [vp]),
        "vox_tile_shape": (i32, [vp, ctypes.POINTER(i32)]),
        "vox_run_sparse": (i32, [vp, vp, vp, sz, vp, vp, i64]),
        "vox_sparse_status": (i32, [vp, vp, vp, ctypes.POINTER(i64)]),
        "vox_pipe_submit_sparse": (i32, [vp, vp, i64, vp, i64, vp, vp, vp, i64, ctypes.POINTER(i64)]),
        "vox_pipe_tile_shape": (i32, [vp, ctypes.POINTER(i32)]),
        "vox_pipe_reserve_pairs": (i32, [vp, i64]),
        "vox_occupancy": (i32, [vp, vp, i32, i32, i32, i32, i32, vp]),
        "vox_lattice": (i32, [vp, vp, i32, i32, i32, vp]),
        "vox_pipe_submit_lattice": (i32, [vp, vp, i32, i32, i32, vp, vp, vp, i64, ctypes.POINTER(i64)]),
        "vox_kernel_launches": (ctypes.c_uint64, []),
        "vox_debug_check_status": (i32, [ctypes.POINTER(ctypes.c_uint32)]),
        "vox_run_noalloc": (i32, [vp, vp, vp, ctypes.POINTER(i64)]),
        "vox_path": (i32, [vp]),
        "vox_debug_selftest": (i32, [vp, i32, vp, vp, i64, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _strerror(code):
    try:
        return load_library().vox_strerror(code).decode()
    except Exception:  # pragma: no cover
        return "error"


def _torch_cuda():
    import torch

    if not torch.cuda.is_available():
        raise RuntimeError("paper_2106_01326_b200 needs a CUDA device: there is no CPU fallback")
    return torch


def _stream_ptr(torch, stream):
    s = stream if stream is not None else torch.cuda.current_stream()
    return ctypes.c_void_p(s.cuda_stream)


class Voxelizer:
    """vox_create / vox_tets / vox_run with torch tensors as device memory.

    verts int32[V][3], tets int32[T][4] and tet_offsets int64[batch+1] are CUDA
    tensors borrowed by the library; run() returns a uint32-as-int32 CUDA tensor
    of shape [batch][nz][ny][nx/32] (layout: include/vox.h).
    """

    def __init__(self, grid, extent=(65536, 65536, 65536), batch=1, tile=None, variant=0):
        self._lib = load_library()
        self._ctx = ctypes.c_void_p()
        self.grid = tuple(int(g) for g in grid)
        self.extent = tuple(int(e) for e in extent)
        self.batch = int(batch)
        rc = self._lib.vox_create(ctypes.byref(self._ctx), *self.grid, *self.extent, self.batch)
        if rc:
            raise VoxError(rc, "vox_create")
        if tile is not None:
            self._ck(self._lib.vox_set_tile(self._ctx, int(tile[0]), int(tile[1])), "vox_set_tile")
        if variant:
            self._ck(self._lib.vox_set_variant(self._ctx, int(variant)), "vox_set_variant")
        self._keep = None
        self._ws = None
        self._out = None
        self._generation = 0  # bumped whenever the mesh or the workspace is re-bound (CapturedStep checks it)

    def _ck(self, rc, where):
        if rc:
            raise VoxError(rc, where, self._lib.vox_last_error(self._ctx).decode())

    def close(self):
        self._generation += 1
        if self._ctx:
            self._lib.vox_destroy(self._ctx)
            self._ctx = ctypes.c_void_p()

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass

    @property
    def grid_words(self):
        return int(self._lib.vox_grid_words(self._ctx))

    @property
    def workspace_bytes(self):
        return int(self._lib.vox_workspace_bytes(self._ctx))

    @property
    def workspace_fixed_bytes(self):
        return int(self._lib.vox_workspace_fixed_bytes(self._ctx))

    def set_tets(self, verts, tets, tet_offsets=None):
        torch = _torch_cuda()
        assert verts.is_cuda and tets.is_cuda and verts.dtype == torch.int32 and tets.dtype == torch.int32
        assert verts.is_contiguous() and tets.is_contiguous()
        V = verts.numel() // 3
        T = tets.numel() // 4
        off_ptr = None
        if self.batch > 1:
            assert tet_offsets is not None and tet_offsets.is_cuda and tet_offsets.dtype == torch.int64
            assert tet_offsets.numel() == self.batch + 1 and tet_offsets.is_contiguous()
            off_ptr = ctypes.c_void_p(tet_offsets.data_ptr())
        self._ck(
            self._lib.vox_tets(self._ctx, ctypes.c_void_p(verts.data_ptr()), V,
                               ctypes.c_void_p(tets.data_ptr()), T, off_ptr),
            "vox_tets",
        )
        self._keep = (verts, tets, tet_offsets)
        self._generation += 1
        self.T, self.V = T, V

    def set_lattice(self, verts, cells, keep):
        """vox_lattice: verts int32[(cx+1)(cy+1)(cz+1)][3] and keep uint8[cx*cy*cz] CUDA tensors (include/vox.h)."""
        torch = _torch_cuda()
        cx, cy, cz = (int(c) for c in cells)
        assert verts.is_cuda and verts.dtype == torch.int32 and verts.is_contiguous()
        assert keep.is_cuda and keep.dtype == torch.uint8 and keep.is_contiguous()
        assert verts.numel() == self.batch * 3 * (cx + 1) * (cy + 1) * (cz + 1)
        assert keep.numel() == self.batch * cx * cy * cz
        self._ck(self._lib.vox_lattice(self._ctx, ctypes.c_void_p(verts.data_ptr()), cx, cy, cz,
                                       ctypes.c_void_p(keep.data_ptr())), "vox_lattice")
        self._keep = (verts, keep)
        self._generation += 1
        self.T, self.V = self.batch * 6 * cx * cy * cz, self.batch * (cx + 1) * (cy + 1) * (cz + 1)

    def alloc_workspace(self, nbytes=None):
        torch = _torch_cuda()
        n = int(nbytes if nbytes is not None else self.workspace_bytes)
        self._ws = torch.empty(max(n, 256), dtype=torch.uint8, device="cuda")
        self._generation += 1
        return self._ws

    def plan(self, stream=None):
        """Exact workspace sizing (count + scan pre-pass; synchronises).  Returns the pair count."""
        torch = _torch_cuda()
        if self._ws is None or self._ws.numel() < self.workspace_fixed_bytes:
            self.alloc_workspace(self.workspace_fixed_bytes)
        pairs = ctypes.c_int64(0)
        self._ck(
            self._lib.vox_plan(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(self._ws.data_ptr()),
                               self._ws.numel(), ctypes.byref(pairs)),
            "vox_plan",
        )
        if self._ws.numel() < self.workspace_bytes:
            self.alloc_workspace()
        return int(pairs.value)

    def run(self, out=None, stream=None):
        torch = _torch_cuda()
        if self._ws is None:
            self.alloc_workspace()
        if out is None:
            nx, ny, nz = self.grid
            out = torch.empty((self.batch, nz, ny, nx // 32), dtype=torch.int32, device="cuda")
        assert out.is_cuda and out.is_contiguous() and out.numel() == self.grid_words
        self._ck(
            self._lib.vox_run(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(self._ws.data_ptr()),
                              self._ws.numel(), ctypes.c_void_p(out.data_ptr())),
            "vox_run",
        )
        return out

    def run_noalloc(self, out, stream=None, stats=True):
        """vox_run_noalloc: run() on the 4 MiB workspace built into libvox.so instead of a torch tensor.

        For code that is handed its input and output tensors but may not allocate device memory itself: a plug-in
        in an application whose pool owns the whole GPU, a loop that cannot afford the device-wide sync of an
        allocation, a process in which another thread is capturing a graph in global mode.  `out` is therefore
        required (nothing is allocated here either).  Jobs whose workspace_bytes exceed NOALLOC_SCRATCH_BYTES raise
        VoxError(-3) before any GPU work.  All calls on a device share the one built-in array: keep them ordered on
        the GPU (one stream, or events), overlapping calls race.  The first call on a device also looks up the
        array's address; make it before any stream capture.  stats=True waits for the stream and returns the
        vox_status dict, raising VoxError(-3) if pairs were dropped; stats=False only enqueues and returns None."""
        torch = _torch_cuda()
        assert out.is_cuda and out.is_contiguous() and out.numel() == self.grid_words
        st = (ctypes.c_int64 * 4)() if stats else None
        self._ck(self._lib.vox_run_noalloc(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(out.data_ptr()), st),
                 "vox_run_noalloc")
        if st is None:
            return None
        return dict(pairs=int(st[0]), culled=int(st[1]), large_pairs=int(st[2]), nonempty_tiles=int(st[3]))

    def capture(self, out, steps=1, stream=None):
        """CUDA graph of `steps` vox_run calls into `out` (vox_run only enqueues: no sync, no allocation, so it can be
        stream-captured).  Returns a CapturedStep; replay() re-runs the step(s) on the mesh, workspace and output
        bound at capture time and refuses (RuntimeError) once set_tets / set_lattice / alloc_workspace / plan / close
        has re-bound any of them, because the graph has the old pointers and sizes baked in.  Runs inside the capture
        record no timing events (vox_timing_*).  Worth ~6-8 us per step: it removes the launch gaps between the memset
        and the four kernels, which is a sixth of a step on the smallest configs and nothing on the large ones
        (DESIGN.md 8)."""
        torch = _torch_cuda()
        if self._ws is None:
            self.alloc_workspace()
        stream = stream or torch.cuda.Stream()
        with torch.cuda.stream(stream):
            self.run(out, stream)  # warm-up outside the capture
            stream.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=stream):
                for _ in range(int(steps)):
                    self.run(out, stream)
        return CapturedStep(self, g, out)

    @property
    def path(self):
        """vox_path: 'tets' (tet array through K1-K4), 'lattice_binned' or 'lattice_fused' -- what the next run() takes."""
        rc = self._lib.vox_path(self._ctx)
        if rc < 0:
            raise VoxError(rc, "vox_path")
        return ("tets", "lattice_binned", "lattice_fused")[rc]

    @property
    def tile_shape(self):
        """dict(ty, tz, nbx, nby, nbz): the binning tile (32 x ty x tz voxels) and tiles per axis."""
        o = (ctypes.c_int * 5)()
        self._ck(self._lib.vox_tile_shape(self._ctx, o), "vox_tile_shape")
        return dict(ty=o[0], tz=o[1], nbx=o[2], nby=o[3], nbz=o[4])

    def run_sparse(self, capacity_tiles, table=None, payload=None, stream=None):
        """vox_run_sparse: returns (table int32[NB], payload int32[capacity][tz][ty]) CUDA tensors
        (layout: include/vox.h).  sparse_status() gives the number of mixed tiles."""
        torch = _torch_cuda()
        if self._ws is None:
            self.alloc_workspace()
        ts = self.tile_shape
        nb = self.batch * ts["nbx"] * ts["nby"] * ts["nbz"]
        if table is None:
            table = torch.empty(nb, dtype=torch.int32, device="cuda")
        if payload is None:
            payload = torch.empty((max(int(capacity_tiles), 1), ts["tz"], ts["ty"]), dtype=torch.int32, device="cuda")
        assert table.is_cuda and table.numel() == nb and table.is_contiguous() and payload.is_contiguous()
        assert payload.numel() >= int(capacity_tiles) * ts["tz"] * ts["ty"]
        self._ck(
            self._lib.vox_run_sparse(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(self._ws.data_ptr()),
                                     self._ws.numel(), ctypes.c_void_p(table.data_ptr()),
                                     ctypes.c_void_p(payload.data_ptr()), int(capacity_tiles)),
            "vox_run_sparse",
        )
        return table, payload

    def sparse_status(self, stream=None):
        """Synchronises.  dict(mixed_tiles, full_tiles); raises VoxError(-3) if payload tiles were dropped."""
        torch = _torch_cuda()
        o = (ctypes.c_int64 * 2)()
        rc = self._lib.vox_sparse_status(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(self._ws.data_ptr()), o)
        self._last_sparse = dict(mixed_tiles=int(o[0]), full_tiles=int(o[1]))
        self._ck(rc, "vox_sparse_status")
        return self._last_sparse

    def status(self, stream=None):
        """Synchronises.  Returns dict(pairs, culled, large_pairs, nonempty_tiles) of the last run() on this
        workspace; raises on overflow.  (plan() may re-allocate the workspace: call status() after run().)"""
        torch = _torch_cuda()
        st = (ctypes.c_int64 * 4)()
        rc = self._lib.vox_status(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(self._ws.data_ptr()), st)
        self._ck(rc, "vox_status")
        return dict(pairs=int(st[0]), culled=int(st[1]), large_pairs=int(st[2]), nonempty_tiles=int(st[3]))

    def validate(self, stream=None):
        torch = _torch_cuda()
        if self._ws is None:
            self.alloc_workspace()
        self._ck(
            self._lib.vox_validate(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(self._ws.data_ptr()),
                                   self._ws.numel()),
            "vox_validate",
        )

    # -- per-kernel device timing (benchmark instrumentation) -----------------------------
    def timing_enable(self, slots):
        self._ck(self._lib.vox_timing_enable(self._ctx, int(slots)), "vox_timing_enable")

    def timing_read(self, run):
        """dict of milliseconds for a completed run (numbered from timing_enable)."""
        ms = (ctypes.c_float * 5)()
        self._ck(self._lib.vox_timing_read(self._ctx, int(run), ms), "vox_timing_read")
        return dict(k1=ms[0], k2=ms[1], k3=ms[2], k4=ms[3], total=ms[4])

    # -- host-buffer end-to-end path (vox_run_host) ---------------------------------------
    def host_arena_bytes(self, V, T):
        return int(self._lib.vox_host_arena_bytes(self._ctx, int(V), int(T)))

    def run_host(self, h_verts, h_tets, h_out, arena, h_tet_offsets=None, stream=None):
        """h_* are (pinned) CPU tensors; arena is a CUDA uint8 tensor.  Synchronises."""
        torch = _torch_cuda()
        V = h_verts.numel() // 3
        T = h_tets.numel() // 4
        off_ptr = ctypes.c_void_p(h_tet_offsets.data_ptr()) if h_tet_offsets is not None else None
        self._ck(
            self._lib.vox_run_host(self._ctx, _stream_ptr(torch, stream), ctypes.c_void_p(h_verts.data_ptr()), V,
                                   ctypes.c_void_p(h_tets.data_ptr()), T, off_ptr,
                                   ctypes.c_void_p(arena.data_ptr()), arena.numel(),
                                   ctypes.c_void_p(h_out.data_ptr())),
            "vox_run_host",
        )
        return h_out


class CapturedStep:
    """A CUDA graph of vox_run steps (Voxelizer.capture).  The graph holds the mesh pointers, the workspace pointer
    and capacity, the tile and the output pointer as they were at capture time; replay() checks that the Voxelizer
    has not re-bound any of them since."""

    def __init__(self, vz, graph, out):
        self._vz, self.graph, self._out = vz, graph, out  # (keeps the output tensor alive)
        self._generation = vz._generation

    def replay(self):
        if self._vz._generation != self._generation:
            raise RuntimeError("CapturedStep.replay: the Voxelizer's mesh or workspace was re-bound (set_tets / "
                               "set_lattice / alloc_workspace / plan / close) after the capture; capture again")
        self.graph.replay()


class Pipe:
    """vox_pipe_*: transfer-overlapped voxelization of a stream of meshes held in pinned host memory.

    submit() takes pinned CPU tensors (verts int32[V][3], tets int32[T][4], optional offsets
    int64[batch+1]) and a pinned CPU output tensor int32[batch][nz][ny][nx/32]; wait(ticket)
    blocks until that output is complete and returns the run's statistics."""

    def __init__(self, grid, extent=(65536, 65536, 65536), batch=1, depth=3, max_V=0, max_T=0, tile=None, variant=0,
                 max_pairs=None):
        torch = _torch_cuda()
        self._lib = load_library()
        self._p = ctypes.c_void_p()
        self.grid = tuple(int(g) for g in grid)
        self.batch, self.depth = int(batch), int(depth)
        rc = self._lib.vox_pipe_create(ctypes.byref(self._p), *self.grid, *(int(e) for e in extent), self.batch,
                                       self.depth, int(max_V), int(max_T))
        if rc:
            raise VoxError(rc, "vox_pipe_create")
        if tile is not None:
            self._ck(self._lib.vox_pipe_set_tile(self._p, int(tile[0]), int(tile[1])), "vox_pipe_set_tile")
        if variant:
            self._ck(self._lib.vox_pipe_set_variant(self._p, int(variant)), "vox_pipe_set_variant")
        if max_pairs is not None:
            self._ck(self._lib.vox_pipe_reserve_pairs(self._p, int(max_pairs)), "vox_pipe_reserve_pairs")
        self.arena_bytes = int(self._lib.vox_pipe_arena_bytes(self._p))
        self._arena = torch.empty(self.arena_bytes + 256, dtype=torch.uint8, device="cuda")
        base = self._arena.data_ptr()
        self._ck(self._lib.vox_pipe_bind(self._p, ctypes.c_void_p((base + 255) & ~255), self.arena_bytes),
                 "vox_pipe_bind")
        self._keep = {}

    def _ck(self, rc, where):
        if rc:
            raise VoxError(rc, where, self._lib.vox_pipe_last_error(self._p).decode())

    def submit(self, h_verts, h_tets, h_out, h_tet_offsets=None):
        for t in (h_verts, h_tets, h_out) + ((h_tet_offsets,) if h_tet_offsets is not None else ()):
            assert not t.is_cuda and t.is_contiguous() and (t.numel() == 0 or t.is_pinned()), \
                "pipe buffers must be pinned CPU tensors"
        ticket = ctypes.c_int64(-1)
        off_ptr = ctypes.c_void_p(h_tet_offsets.data_ptr()) if h_tet_offsets is not None else None
        self._ck(
            self._lib.vox_pipe_submit(self._p, ctypes.c_void_p(h_verts.data_ptr()), h_verts.numel() // 3,
                                      ctypes.c_void_p(h_tets.data_ptr()), h_tets.numel() // 4, off_ptr,
                                      ctypes.c_void_p(h_out.data_ptr()), ctypes.byref(ticket)),
            "vox_pipe_submit",
        )
        self._keep[ticket.value] = (h_verts, h_tets, h_out, h_tet_offsets)
        return int(ticket.value)

    @property
    def tile_shape(self):
        o = (ctypes.c_int * 5)()
        self._ck(self._lib.vox_pipe_tile_shape(self._p, o), "vox_pipe_tile_shape")
        return dict(ty=o[0], tz=o[1], nbx=o[2], nby=o[3], nbz=o[4])

    def submit_sparse(self, h_verts, h_tets, h_table, h_payload, capacity_tiles, h_tet_offsets=None):
        """Sparse output (include/vox.h): h_table int32[NB] and h_payload int32[capacity][tz][ty] are pinned
        CPU tensors; the kernel stores the mixed tiles straight into h_payload."""
        for t in (h_verts, h_tets, h_table, h_payload) + ((h_tet_offsets,) if h_tet_offsets is not None else ()):
            assert not t.is_cuda and t.is_contiguous() and (t.numel() == 0 or t.is_pinned()), \
                "pipe buffers must be pinned CPU tensors"
        ts = self.tile_shape
        assert h_table.numel() == self.batch * ts["nbx"] * ts["nby"] * ts["nbz"]
        assert h_payload.numel() >= int(capacity_tiles) * ts["ty"] * ts["tz"]
        ticket = ctypes.c_int64(-1)
        off_ptr = ctypes.c_void_p(h_tet_offsets.data_ptr()) if h_tet_offsets is not None else None
        self._ck(
            self._lib.vox_pipe_submit_sparse(self._p, ctypes.c_void_p(h_verts.data_ptr()), h_verts.numel() // 3,
                                             ctypes.c_void_p(h_tets.data_ptr()), h_tets.numel() // 4, off_ptr,
                                             ctypes.c_void_p(h_table.data_ptr()),
                                             ctypes.c_void_p(h_payload.data_ptr()), int(capacity_tiles),
                                             ctypes.byref(ticket)),
            "vox_pipe_submit_sparse",
        )
        self._keep[ticket.value] = (h_verts, h_tets, h_table, h_payload, h_tet_offsets)
        return int(ticket.value)

    def submit_lattice(self, h_verts, cells, h_keep, h_out, h_payload=None, capacity_tiles=-1):
        """vox_pipe_submit_lattice: lattice vertices + keep mask in (pinned); dense grid out (capacity_tiles < 0)
        or tile table + payload (sparse)."""
        bufs = (h_verts, h_keep, h_out) + ((h_payload,) if h_payload is not None else ())
        for t in bufs:
            assert not t.is_cuda and t.is_contiguous() and (t.numel() == 0 or t.is_pinned()), \
                "pipe buffers must be pinned CPU tensors"
        cx, cy, cz = (int(c) for c in cells)
        assert h_verts.numel() == self.batch * 3 * (cx + 1) * (cy + 1) * (cz + 1)
        assert h_keep.numel() == self.batch * cx * cy * cz
        ticket = ctypes.c_int64(-1)
        self._ck(
            self._lib.vox_pipe_submit_lattice(self._p, ctypes.c_void_p(h_verts.data_ptr()), cx, cy, cz,
                                              ctypes.c_void_p(h_keep.data_ptr()), ctypes.c_void_p(h_out.data_ptr()),
                                              ctypes.c_void_p(h_payload.data_ptr()) if h_payload is not None else None,
                                              int(capacity_tiles), ctypes.byref(ticket)),
            "vox_pipe_submit_lattice",
        )
        self._keep[ticket.value] = bufs
        return int(ticket.value)

    def wait(self, ticket):
        st = (ctypes.c_int64 * 6)()
        rc = self._lib.vox_pipe_wait(self._p, int(ticket), st)
        self._keep.pop(int(ticket), None)
        self.last_stats = dict(pairs=int(st[0]), culled=int(st[1]), large_pairs=int(st[2]), nonempty_tiles=int(st[3]),
                               mixed_tiles=int(st[4]), full_tiles=int(st[5]))
        self._ck(rc, "vox_pipe_wait")
        return self.last_stats

    def close(self):
        if self._p:
            self._lib.vox_pipe_destroy(self._p)
            self._p = ctypes.c_void_p()
        self._arena = None

    def __del__(self):  # pragma: no cover
        try:
            self.close()
        except Exception:
            pass


def voxelize(verts, tets, grid, extent=(65536, 65536, 65536), tet_offsets=None, tile=None, variant=0, exact_plan=True):
    """One-shot: numpy/torch in, numpy uint32[batch][nz][ny][nx/32] out (device path, via vox_run)."""
    torch = _torch_cuda()
    import numpy as np

    def dev(a, dt):
        if isinstance(a, torch.Tensor):
            return a.to(device="cuda", dtype=dt).contiguous()
        return torch.from_numpy(np.ascontiguousarray(a)).to(device="cuda", dtype=dt).contiguous()

    v = dev(verts, torch.int32).reshape(-1, 3)
    t = dev(tets, torch.int32).reshape(-1, 4)
    batch = 1 if tet_offsets is None else len(tet_offsets) - 1
    off = dev(tet_offsets, torch.int64) if tet_offsets is not None else None
    vz = Voxelizer(grid, extent, batch, tile=tile, variant=variant)
    try:
        vz.set_tets(v, t, off)
        if exact_plan:
            vz.plan()
        out = vz.run()
        vz.last_status = vz.status()
        res = out.cpu().numpy().view(np.uint32)
        voxelize.last_status = vz.last_status
        return res
    finally:
        vz.close()


def occupancy(bits_fine, grid, k, batch=1, out=None, stream=None):
    """vox_occupancy: fold a bit grid voxelized at k times `grid`'s resolution (CUDA int32 tensor
    [batch][k*nz][k*ny][k*nx/32]) into solid sub-sample counts, CUDA uint8 [batch][nz][ny][nx]."""
    torch = _torch_cuda()
    lib = load_library()
    nx, ny, nz = (int(g) for g in grid)
    assert bits_fine.is_cuda and bits_fine.is_contiguous()
    assert bits_fine.numel() == batch * (k * nz) * (k * ny) * (k * nx // 32)
    if out is None:
        out = torch.empty((batch, nz, ny, nx), dtype=torch.uint8, device="cuda")
    rc = lib.vox_occupancy(_stream_ptr(torch, stream), ctypes.c_void_p(bits_fine.data_ptr()), nx, ny, nz, int(batch),
                           int(k), ctypes.c_void_p(out.data_ptr()))
    if rc:
        raise VoxError(rc, "vox_occupancy")
    return out


def voxelize_host(verts, tets, grid, extent=(65536, 65536, 65536), tet_offsets=None):
    """One-shot through vox_run_host (host buffers in, host grid out)."""
    torch = _torch_cuda()
    import numpy as np

    hv = torch.from_numpy(np.ascontiguousarray(verts, dtype=np.int32)).pin_memory()
    ht = torch.from_numpy(np.ascontiguousarray(tets, dtype=np.int32)).pin_memory()
    batch = 1 if tet_offsets is None else len(tet_offsets) - 1
    ho = torch.from_numpy(np.ascontiguousarray(tet_offsets, dtype=np.int64)).pin_memory() if batch > 1 else None
    vz = Voxelizer(grid, extent, batch)
    try:
        nx, ny, nz = vz.grid
        out = torch.empty((batch, nz, ny, nx // 32), dtype=torch.int32).pin_memory()
        arena = torch.empty(vz.host_arena_bytes(hv.numel() // 3, ht.numel() // 4), dtype=torch.uint8, device="cuda")
        vz.run_host(hv, ht, out, arena, ho)
        return out.numpy().view(np.uint32)
    finally:
        vz.close()


def debug_check_status():
    """vox_debug_check_status: (checks_compiled_in, code of the first violated check or 0).  Synchronises the device."""
    code = ctypes.c_uint32(0)
    rc = load_library().vox_debug_check_status(ctypes.byref(code))
    if rc < 0:
        raise VoxError(rc, "vox_debug_check_status")
    return bool(rc), int(code.value)


def kernel_launches() -> int:
    """vox_kernel_launches: kernels launched by libvox.so in this process so far."""
    return int(load_library().vox_kernel_launches())


def probe_int32(kind=0, blocks=148 * 16, iters=4096, repeats=5):
    """Measured INT32 throughput (thread-ops/s) of the probe kernel; CUDA events on the current stream."""
    torch = _torch_cuda()
    lib = load_library()
    sink = torch.zeros(4, dtype=torch.int32, device="cuda")
    ops = ctypes.c_double(0)
    st = _stream_ptr(torch, None)
    best = None
    for _ in range(repeats + 1):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        rc = lib.vox_probe_int32(st, kind, blocks, iters, ctypes.c_void_p(sink.data_ptr()), ctypes.byref(ops))
        if rc:
            raise VoxError(rc, "vox_probe_int32")
        e1.record()
        e1.synchronize()
        ms = e0.elapsed_time(e1)
        best = ms if best is None else min(best, ms)
    return ops.value / (best * 1e-3)
