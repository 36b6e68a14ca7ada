"""Thin ctypes binding of libreshard.so (include/reshard.h): argument marshalling only.

Every step of the path runs inside the library: the planner in C++ on the host, the data path in
the sm_100a kernels.  There is no Python or CPU fallback: if the library is missing, loading
fails; if no CUDA device is present, reshard_plan without RS_HOST_ONLY fails with RS_ECUDA.

Function names mirror the C ABI:  reshard_plan -> Plan(...), reshard_execute -> Plan.execute, ...
Device buffers are passed as integer addresses (e.g. torch.Tensor.data_ptr()); streams as the
integer cudaStream_t (torch.cuda.current_stream().cuda_stream).
"""
import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libreshard.so")

RS_OK, RS_EINVAL, RS_ESPEC, RS_EDIVIS, RS_EUNSUPPORTED, RS_ENOMEM, RS_ECUDA = range(7)
RS_LB_GREEDY, RS_LB_NAIVE = 0x0, 0x1
RS_PATH_AUTO, RS_PATH_LSU, RS_PATH_BULK, RS_PATH_BULK_SHIFT, RS_PATH_TMAP = 0x00, 0x10, 0x20, 0x30, 0x40
RS_HOST_ONLY = 0x100
RS_EVEN_ONLY = 0x200
RS_WITH_STRATEGIES = 0x400
RS_OP_SENDRECV, RS_OP_AG_SCATTER, RS_OP_AG_GATHER, RS_OP_AGL_SCATTER, RS_OP_AGL_GATHER = 4, 5, 6, 7, 8
RS_STRATEGY_BROADCAST, RS_STRATEGY_SENDRECV, RS_STRATEGY_ALLGATHER, RS_STRATEGY_ALLGATHER_LOCAL = 0, 1, 2, 3
RS_OP_EXECUTE, RS_OP_PACK, RS_OP_UNPACK, RS_OP_EXECUTE_SLABS = 0, 1, 2, 3
RS_SRC, RS_DST = 0, 1
RS_SCHED_NONE, RS_SCHED_NAIVE, RS_SCHED_LOAD_BALANCE, RS_SCHED_DFS, RS_SCHED_GREEDY, RS_SCHED_ENSEMBLE = range(6)
RS_MAX_NDIM, RS_MAX_MESH_NDIM, RS_MAX_DEVICES = 8, 4, 128

# every symbol include/reshard.h declares (tests check the library exports exactly these)
SYMBOLS = [
    "reshard_plan", "reshard_plan_ex", "reshard_plan_group", "reshard_plan_schedule", "reshard_plan_destroy", "reshard_plan_info", "reshard_op_info", "reshard_op_tables", "reshard_op_tiles",
    "reshard_plan_local_shape", "reshard_plan_device_box", "reshard_plan_slice", "reshard_plan_sender_bytes",
    "reshard_plan_message", "reshard_execute", "reshard_execute_static", "reshard_execute_strategy", "reshard_pack", "reshard_unpack", "reshard_execute_host",
    "reshard_ipc_export", "reshard_ipc_import", "reshard_ipc_release_all",
    "reshard_host_workspace_bytes", "reshard_pipeline_simulate", "reshard_pipeline_least_delay", "reshard_launch_count", "reshard_strerror", "reshard_last_error",
    "reshard_version",
]


class PlanInfo(C.Structure):
    _fields_ = [("ndim", C.c_int32), ("elem_bytes", C.c_int32), ("n_src", C.c_int32), ("n_dst", C.c_int32),
                ("n_slices", C.c_int32), ("n_messages", C.c_int32),
                ("tensor_bytes", C.c_int64), ("src_shard_bytes", C.c_int64), ("dst_shard_bytes", C.c_int64),
                ("unique_read_bytes", C.c_int64), ("write_bytes", C.c_int64), ("max_sender_bytes", C.c_int64),
                ("arena_bytes", C.c_int64), ("lb_mode", C.c_int32), ("device", C.c_int32)]


class OpInfo(C.Structure):
    _fields_ = [("path", C.c_int32), ("vec_bytes", C.c_int32), ("n_tasks", C.c_int32), ("n_dsts", C.c_int32),
                ("n_tiles", C.c_int32), ("tile_bytes", C.c_int32), ("grid", C.c_int32), ("block", C.c_int32),
                ("smem_bytes", C.c_int32), ("read_bytes", C.c_int64), ("write_bytes", C.c_int64),
                ("min_run_bytes", C.c_int64), ("n_segs", C.c_int32), ("table_bytes", C.c_int32), ("pace_permille", C.c_int32),
                ("reserved", C.c_int32)]


class Tuning(C.Structure):
    """rs_tuning: launch-shape overrides for tests and sweeps (0 = the library's choice)"""
    _fields_ = [("bulk_warps", C.c_int32), ("bulk_stages", C.c_int32), ("bulk_lookahead", C.c_int32),
                ("bulk_tile_bytes", C.c_int32), ("bulk_ctas", C.c_int32), ("bulk_ctas_mcast", C.c_int32),
                ("shift_warps", C.c_int32), ("shift_stages", C.c_int32), ("shift_lookahead", C.c_int32),
                ("shift_tile_bytes", C.c_int32), ("lsu_tile_bytes", C.c_int32), ("lsu_ctas_per_sm", C.c_int32),
                ("task_order", C.c_int32), ("small_op_bytes_mib", C.c_int32), ("tiles_per_worker", C.c_int32), ("pace_permille", C.c_int32), ("no_pdl", C.c_int32),
                ("pace_burst", C.c_int32), ("pace_adapt", C.c_int32), ("ring_min_smem", C.c_int32), ("lsu_narrow", C.c_int32), ("shift_mode", C.c_int32)]


class PlanOpts(C.Structure):
    _fields_ = [("flags", C.c_uint32), ("schedule", C.c_int32), ("src_devices_per_host", C.c_int32),
                ("dst_devices_per_host", C.c_int32), ("trials", C.c_int32), ("max_ctas", C.c_int32),
                ("node_budget", C.c_int64), ("seed", C.c_uint64), ("tuning", C.POINTER(Tuning)),
                ("src_owner", C.POINTER(C.c_int32)), ("rank", C.c_int32), ("reserved", C.c_int32)]


class ScheduleInfo(C.Structure):
    _fields_ = [("algorithm", C.c_int32), ("winner", C.c_int32), ("n_tasks", C.c_int32), ("n_rounds", C.c_int32),
                ("n_src_hosts", C.c_int32), ("n_dst_hosts", C.c_int32), ("dfs_finished", C.c_int32),
                ("reserved", C.c_int32), ("dfs_nodes", C.c_int64), ("makespan", C.c_int64),
                ("busiest_host_bytes", C.c_int64)]


RS_PIPE_MAX_STAGES = 64
RS_PIPE_1F1B, RS_PIPE_EAGER_1F1B = 0, 1
RS_PIPE_F, RS_PIPE_B, RS_PIPE_BA, RS_PIPE_BW = 0, 1, 2, 3


class PipelineOpts(C.Structure):
    _fields_ = [("schedule", C.c_int32), ("n_stages", C.c_int32), ("n_micro_batches", C.c_int32), ("overlap", C.c_int32),
                ("bw_delay", C.c_int32), ("reserved", C.c_int32), ("fwd", C.POINTER(C.c_int64)), ("bwd", C.POINTER(C.c_int64)),
                ("bwd_act", C.POINTER(C.c_int64)), ("comm_fwd", C.c_int64), ("comm_bwd", C.c_int64)]


class PipelineResult(C.Structure):
    _fields_ = [("makespan", C.c_int64), ("ops_per_stage", C.c_int32), ("reserved", C.c_int32),
                ("warmup", C.c_int32 * RS_PIPE_MAX_STAGES), ("peak_activations", C.c_int32 * RS_PIPE_MAX_STAGES),
                ("busy", C.c_int64 * RS_PIPE_MAX_STAGES)]


class ReshardError(RuntimeError):
    def __init__(self, code, text):
        super().__init__("reshard: %s (%s)" % (text, _lib().reshard_strerror(code).decode()))
        self.code = code


_LIB = None


def _lib():
    global _LIB
    if _LIB is None:
        try:                                  # build in-tree if missing or older than its sources (nvcc, sm_100a only)
            from . import build as _build
            _build.build()
        except Exception as ex:               # noqa: BLE001 -- no nvcc, or a compile error: say so, there is no fallback
            if not os.path.exists(LIB_PATH) or _build._stale():      # an up-to-date library needs no compiler
                raise ImportError("libreshard.so is missing or older than its sources and could not be built (%s): run "
                                  "`python -m paper_2211_05322_b200.build` (there is no fallback path)" % ex)
        try:
            L = C.CDLL(LIB_PATH)
        except OSError:                      # libcudart not on the loader path: torch ships one
            import torch  # noqa: F401
            L = C.CDLL(LIB_PATH)
        for name in SYMBOLS:
            getattr(L, name).restype = C.c_int
        L.reshard_plan_destroy.restype = None
        L.reshard_host_workspace_bytes.restype = C.c_int64
        L.reshard_launch_count.restype = C.c_int64
        for name in ("reshard_strerror", "reshard_last_error", "reshard_version"):
            getattr(L, name).restype = C.c_char_p
        _LIB = L
    return _LIB


def _chk(rc):
    if rc != RS_OK:
        raise ReshardError(rc, _lib().reshard_last_error().decode() or "error %d" % rc)


def _i64(xs):
    return (C.c_int64 * len(xs))(*[int(x) for x in xs])


def _i32(xs):
    return (C.c_int32 * len(xs))(*[int(x) for x in xs])


def _ptrs(addrs):
    return (C.c_void_p * len(addrs))(*[C.c_void_p(int(a) if a else None) for a in addrs])


RS_IPC_HANDLE_BYTES = 80


def ipc_export(dev_ptr):
    """reshard_ipc_export: bytes to send to the peers for a device pointer of this process"""
    buf = C.create_string_buffer(RS_IPC_HANDLE_BYTES)
    _chk(_lib().reshard_ipc_export(C.c_void_p(int(dev_ptr)), buf))
    return buf.raw


def ipc_import(handle):
    """reshard_ipc_import: device pointer, valid in this process, of another process's exported pointer"""
    out = C.c_void_p()
    _chk(_lib().reshard_ipc_import(C.create_string_buffer(bytes(handle), RS_IPC_HANDLE_BYTES), C.byref(out)))
    return int(out.value)


def ipc_release_all():
    _chk(_lib().reshard_ipc_release_all())


def version():
    return _lib().reshard_version().decode()


def launch_count():
    return int(_lib().reshard_launch_count())


class Plan:
    """reshard_plan(...) handle.  See include/reshard.h for the contract of every call."""

    def __init__(self, global_shape, elem_bytes, src_mesh, src_spec, dst_mesh, dst_spec, flags=0, opts=None):
        """opts: dict of rs_plan_opts fields (schedule, src_devices_per_host, ..., tuning=dict of rs_tuning
        fields) -> reshard_plan_ex"""
        self._h = C.c_void_p()
        if opts is None:
            _chk(_lib().reshard_plan(_i64(global_shape), len(global_shape), int(elem_bytes),
                                     _i32(src_mesh), len(src_mesh), src_spec.encode(),
                                     _i32(dst_mesh), len(dst_mesh), dst_spec.encode(),
                                     C.c_uint32(flags), C.byref(self._h)))
        else:
            opts = dict(opts)
            tune = opts.pop("tuning", None)
            owner = opts.pop("src_owner", None)
            o = PlanOpts(flags=flags, **opts)
            if owner is not None:                                    # multi-process executor: rank = opts["rank"]
                arr = _i32(owner)
                o.src_owner = C.cast(arr, C.POINTER(C.c_int32))
            if tune:
                t = Tuning(**tune)                                   # the plan copies it
                o.tuning = C.pointer(t)
            _chk(_lib().reshard_plan_ex(_i64(global_shape), len(global_shape), int(elem_bytes),
                                        _i32(src_mesh), len(src_mesh), src_spec.encode(),
                                        _i32(dst_mesh), len(dst_mesh), dst_spec.encode(),
                                        C.byref(o), C.byref(self._h)))
        self.info = PlanInfo()
        _chk(_lib().reshard_plan_info(self._h, C.byref(self.info)))
        self.ndim = self.info.ndim

    @classmethod
    def group(cls, plans, flags=0):
        """reshard_plan_group: one plan whose execute() runs all of `plans` in a single launch; its pointer lists
        are the concatenations of the members' lists"""
        self = cls.__new__(cls)
        self._h = C.c_void_p()
        arr = (C.c_void_p * len(plans))(*[p._h for p in plans])
        _chk(_lib().reshard_plan_group(arr, len(plans), C.c_uint32(flags), C.byref(self._h)))
        self.info = PlanInfo()
        _chk(_lib().reshard_plan_info(self._h, C.byref(self.info)))
        self.ndim = 0
        return self

    def close(self):
        if getattr(self, "_h", None) and _LIB is not None:     # _LIB is None again while the interpreter shuts down
            _LIB.reshard_plan_destroy(self._h)
            self._h = None

    __del__ = close

    # ---- queries
    def op_info(self, op):
        out = OpInfo()
        _chk(_lib().reshard_op_info(self._h, op, C.byref(out)))
        return out

    def op_tables(self, op):
        """raw bytes of (tasks, dsts, segs); layouts in csrc/tables.h"""
        oi = self.op_info(op)
        t, d, g = (C.create_string_buffer(max(1, oi.n_tasks * 224)), C.create_string_buffer(max(1, oi.n_dsts * 16)),
                   C.create_string_buffer(max(1, oi.n_segs * 16)))
        _chk(_lib().reshard_op_tables(self._h, op, t, d, g))
        return t.raw[:oi.n_tasks * 224], d.raw[:oi.n_dsts * 16], g.raw[:oi.n_segs * 16]

    def op_tiles(self, op, first=0, count=None):
        """raw bytes of tiles first .. first + count - 1 as the LIBRARY decodes them (32-byte RsTile records)"""
        if count is None:
            count = self.op_info(op).n_tiles - first
        buf = C.create_string_buffer(max(1, count * 32))
        _chk(_lib().reshard_op_tiles(self._h, op, C.c_int64(first), C.c_int64(count), buf))
        return buf.raw[:count * 32]

    def local_shape(self, side):
        out = (C.c_int64 * self.ndim)()
        _chk(_lib().reshard_plan_local_shape(self._h, side, out))
        return tuple(out)

    def device_box(self, side, dev):
        lo, hi = (C.c_int64 * self.ndim)(), (C.c_int64 * self.ndim)()
        _chk(_lib().reshard_plan_device_box(self._h, side, dev, lo, hi))
        return tuple(lo), tuple(hi)

    def slice(self, i):
        lo, hi = (C.c_int64 * self.ndim)(), (C.c_int64 * self.ndim)()
        sender, ns, nr = C.c_int32(), C.c_int32(), C.c_int32()
        senders, receivers = (C.c_int32 * self.info.n_src)(), (C.c_int32 * self.info.n_dst)()
        _chk(_lib().reshard_plan_slice(self._h, i, lo, hi, C.byref(sender), C.byref(ns), senders, C.byref(nr),
                                       receivers))
        return dict(lo=tuple(lo), hi=tuple(hi), sender=sender.value, senders=list(senders[:ns.value]),
                    receivers=list(receivers[:nr.value]))

    def slices(self):
        return [self.slice(i) for i in range(self.info.n_slices)]

    def schedule(self):
        """reshard_plan_schedule -> dict(info=ScheduleInfo, sender_host, start, order)"""
        n = self.info.n_slices
        info, sh, st, od = ScheduleInfo(), (C.c_int32 * n)(), (C.c_int64 * n)(), (C.c_int32 * n)()
        _chk(_lib().reshard_plan_schedule(self._h, C.byref(info), sh, st, od))
        return dict(info=info, sender_host=list(sh), start=list(st), order=list(od))

    def sender_bytes(self):
        out = (C.c_int64 * self.info.n_src)()
        _chk(_lib().reshard_plan_sender_bytes(self._h, out))
        return list(out)

    def message(self, m):
        s, r, n = C.c_int32(), C.c_int32(), C.c_int32()
        off, nb = C.c_int64(), C.c_int64()
        ids = (C.c_int32 * self.info.n_slices)()
        _chk(_lib().reshard_plan_message(self._h, m, C.byref(s), C.byref(r), C.byref(off), C.byref(nb), C.byref(n), ids))
        return dict(sender=s.value, receiver=r.value, offset=off.value, bytes=nb.value, slice_ids=list(ids[:n.value]))

    def messages(self):
        return [self.message(m) for m in range(self.info.n_messages)]

    def host_workspace_bytes(self):
        return int(_lib().reshard_host_workspace_bytes(self._h))

    # ---- data path (device addresses in, nothing out; asynchronous on `stream`)
    def execute(self, src_ptrs, dst_ptrs, stream=0):
        _chk(_lib().reshard_execute(self._h, _ptrs(src_ptrs), _ptrs(dst_ptrs), C.c_void_p(stream)))

    def execute_static(self, src_ptrs, dst_ptrs, stream=0):
        """reshard_execute_static: no device allocation anywhere (works on RS_HOST_ONLY plans); tables in the library's static device array"""
        _chk(_lib().reshard_execute_static(self._h, _ptrs(src_ptrs), _ptrs(dst_ptrs), C.c_void_p(stream)))

    def execute_strategy(self, strategy, src_ptrs, dst_ptrs, stream=0):
        _chk(_lib().reshard_execute_strategy(self._h, int(strategy), _ptrs(src_ptrs), _ptrs(dst_ptrs), C.c_void_p(stream)))

    def pack(self, src_ptrs, arena_ptr, stream=0):
        _chk(_lib().reshard_pack(self._h, _ptrs(src_ptrs), C.c_void_p(arena_ptr), C.c_void_p(stream)))

    def unpack(self, arena_ptr, dst_ptrs, stream=0):
        _chk(_lib().reshard_unpack(self._h, C.c_void_p(arena_ptr), _ptrs(dst_ptrs), C.c_void_p(stream)))

    def execute_host(self, src_host_ptrs, dst_host_ptrs, workspace_ptr, stream=0):
        """returns (h2d_bytes, d2h_bytes)"""
        up, down = C.c_int64(), C.c_int64()
        _chk(_lib().reshard_execute_host(self._h, _ptrs(src_host_ptrs), _ptrs(dst_host_ptrs),
                                         C.c_void_p(workspace_ptr), C.c_void_p(stream), C.byref(up), C.byref(down)))
        return up.value, down.value


def pipeline_simulate(schedule, n_stages, n_micro_batches, fwd, bwd, comm_fwd, comm_bwd, overlap=True, bwd_act=None,
                      bw_delay=0):
    """reshard_pipeline_simulate -> dict(makespan, warmup, peak, busy, ops=[per stage list of (kind, micro, start, end)]).
    fwd / bwd / bwd_act: one int (every stage) or a list per stage."""
    def per_stage(x):
        return _i64(x if isinstance(x, (list, tuple)) else [x] * n_stages)
    f, b = per_stage(fwd), per_stage(bwd)
    ba = per_stage(bwd_act) if bwd_act is not None else None
    o = PipelineOpts(schedule=schedule, n_stages=n_stages, n_micro_batches=n_micro_batches, overlap=int(bool(overlap)),
                     bw_delay=bw_delay, fwd=f, bwd=b, bwd_act=ba, comm_fwd=comm_fwd, comm_bwd=comm_bwd)
    res = PipelineResult()
    _chk(_lib().reshard_pipeline_simulate(C.byref(o), C.byref(res), None, None, None, None))
    n = n_stages * res.ops_per_stage
    kind, micro, start, end = (C.c_int32 * n)(), (C.c_int32 * n)(), (C.c_int64 * n)(), (C.c_int64 * n)()
    _chk(_lib().reshard_pipeline_simulate(C.byref(o), C.byref(res), kind, micro, start, end))
    k = res.ops_per_stage
    ops = [[(kind[i * k + j], micro[i * k + j], start[i * k + j], end[i * k + j]) for j in range(k)] for i in range(n_stages)]
    return dict(makespan=res.makespan, warmup=list(res.warmup[:n_stages]), peak=list(res.peak_activations[:n_stages]),
                busy=list(res.busy[:n_stages]), ops=ops)


def pipeline_least_delay(schedule, n_stages, stage, n_micro_batches, fwd, bwd, bwd_act, comm_bwd):
    return int(_lib().reshard_pipeline_least_delay(schedule, n_stages, stage, n_micro_batches, C.c_int64(fwd), C.c_int64(bwd),
                                                   C.c_int64(bwd_act), C.c_int64(comm_bwd)))
