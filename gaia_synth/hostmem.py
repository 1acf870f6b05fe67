"""How much host memory a test or a bench leg may take: the smaller of what the kernel reports as available and
what the process's memory cgroup (v2 or v1) still allows.  psutil alone does not see a cgroup limit, and a copy of
C4 to the host (112 GB) that crosses it gets the whole process killed instead of a skip."""
import os


def _read_int(path):
    try:
        with open(path) as f:
            t = f.read().strip()
        return None if t in ("", "max") else int(t)
    except (OSError, ValueError):
        return None


def _cgroup_headroom():
    """Bytes left under the tightest memory limit of this process's cgroup chain, or None if there is no limit."""
    best = None
    paths = []
    try:
        with open("/proc/self/cgroup") as f:
            for line in f:
                parts = line.strip().split(":", 2)
                if len(parts) != 3:
                    continue
                _, ctrl, rel = parts
                if ctrl == "":                                    # cgroup v2
                    base, lim, cur = "/sys/fs/cgroup", "memory.max", "memory.current"
                elif "memory" in ctrl.split(","):                 # cgroup v1
                    base, lim, cur = "/sys/fs/cgroup/memory", "memory.limit_in_bytes", "memory.usage_in_bytes"
                else:
                    continue
                rel = rel.strip("/")
                # the group itself and every ancestor up to the mount point (a container usually sees its own
                # group AT the mount point, so the root entry matters too)
                chain = [""]
                acc = ""
                for piece in [p for p in rel.split("/") if p]:
                    acc = acc + "/" + piece
                    chain.append(acc)
                for c in chain:
                    paths.append((base + c + "/" + lim, base + c + "/" + cur))
    except OSError:
        return None
    for lim_p, cur_p in paths:
        lim = _read_int(lim_p)
        if lim is None or lim <= 0 or lim >= (1 << 60):           # "max" / the v1 no-limit sentinel
            continue
        cur = _read_int(cur_p) or 0
        room = max(0, lim - cur)
        best = room if best is None else min(best, room)
    return best


def available_host_memory(default=16 << 30):
    """Bytes of host memory that can still be taken (MemAvailable, capped by the cgroup's headroom)."""
    avail = None
    try:
        import psutil
        avail = int(psutil.virtual_memory().available)
    except Exception:
        try:
            with open("/proc/meminfo") as f:
                for line in f:
                    if line.startswith("MemAvailable:"):
                        avail = int(line.split()[1]) * 1024
                        break
        except OSError:
            pass
    if avail is None:
        avail = default
    room = _cgroup_headroom()
    if room is not None:
        avail = min(avail, room)
    return avail


def host_threads():
    """CPU threads this process may run on (affinity / cpuset aware)."""
    try:
        return len(os.sched_getaffinity(0))
    except (AttributeError, OSError):
        return os.cpu_count() or 1
