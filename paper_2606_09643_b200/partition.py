"""Spatial partitioning of the GPU between co-resident backbones.

PAPER.md L253: "When multiple FM instances share a single accelerator, FMplex assigns their CUDA streams to disjoint Thread
Processing Cluster (TPC) subsets."  On B200 the supported mechanism is a CUDA green context: the device's SMs are split into
disjoint groups, each group backs a green context, and a stream created in it runs its kernels on that group's SMs only.
libfmx needs nothing special: fmx_forward_mixed takes the stream; its persistent kernels size their grids by the whole device and
simply take more waves on a partition.  (FMX_OPT_SHRINK_FUSED must stay off: it assumes every CTA pair is resident at once.)

Marshalling only (driver API through cuda-python); no arithmetic of the method.
"""
from cuda.bindings import driver as drv


def _ck(r):
    if r[0] != drv.CUresult.CUDA_SUCCESS:
        raise RuntimeError(f"CUDA driver call failed: {r[0]}")
    return r[1:] if len(r) > 2 else (r[1] if len(r) == 2 else None)


class SmPartition:
    """Two disjoint SM groups of one device: `first_sms` SMs (rounded by the driver to its granularity) and the rest.
    .streams = (raw CUstream handle on the first group, raw handle on the second); .sm_counts = their SM counts."""

    def __init__(self, device=0, first_sms=64):
        dev = _ck(drv.cuDeviceGet(device))
        res = _ck(drv.cuDeviceGetDevResource(dev, drv.CUdevResourceType.CU_DEV_RESOURCE_TYPE_SM))
        groups, n, rest = _ck(drv.cuDevSmResourceSplitByCount(1, res, 0, first_sms))
        if n != 1 or rest.sm.smCount == 0:
            raise RuntimeError("the device's SMs could not be split into two groups")
        self.sm_counts = (int(groups[0].sm.smCount), int(rest.sm.smCount))
        self._green = []
        self.streams = []
        for r in (groups[0], rest):
            desc = _ck(drv.cuDevResourceGenerateDesc([r], 1))
            g = _ck(drv.cuGreenCtxCreate(desc, dev, drv.CUgreenCtxCreate_flags.CU_GREEN_CTX_DEFAULT_STREAM))
            self._green.append(g)
            self.streams.append(int(_ck(drv.cuGreenCtxStreamCreate(g, drv.CUstream_flags.CU_STREAM_NON_BLOCKING, 0))))

    def close(self):
        for s in self.streams:
            drv.cuStreamDestroy(s)
        for g in self._green:
            drv.cuGreenCtxDestroy(g)
        self.streams, self._green = [], []
