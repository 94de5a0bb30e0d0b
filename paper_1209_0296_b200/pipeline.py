"""Host-buffer pipeline over the C ABI: upload a configuration, sweep it, download the (B, M) series -- step after step,
with the upload of step k+1 overlapping the sweeps of step k.

This is the sequence `bench.py` times as `e2e` and the sequence `tests/test_gpu_e2e.py` holds to the oracle; it lives
here so that both run the same code.  Marshalling and stream ordering only: every copy and every kernel is enqueued
by a liblsm call (lsm_stage_spins_host, lsm_set_spins, lsm_sweep_record_host_async).

Per step k (b = k & 1; two staging buffers, two device series buffers, two pinned host series buffers):
  copy stream   : h_in[k] -> d_stage[b]                         (after set_spins of step k-2 has consumed d_stage[b])
  compute stream: wait for that copy; lsm_set_spins(d_stage[b], t_k); S sweeps recording into d_obs[b];
                  d_obs[b] -> h_obs[b] (device -> pinned host)
  host          : before step k reuses h_obs[b], wait for step k-2's download and hand its series to `consume`.
"""
from __future__ import annotations


class HostPipeline:
    def __init__(self, lat, sweeps_per_step: int):
        import torch

        self.lat, self.S = lat, int(sweeps_per_step)
        dev, N, S = lat.device, lat.N, self.S
        with torch.cuda.device(dev):
            self.h_obs = [torch.empty((S, 2), dtype=torch.int64).pin_memory() for _ in range(2)]
            self.d_obs = [torch.empty((S, 2), dtype=torch.int64, device=dev) for _ in range(2)]
            self.d_stage = [torch.empty(N, dtype=torch.int8, device=dev) for _ in range(2)]
            self.copy_stream = torch.cuda.Stream(device=dev)
            self.staged = [torch.cuda.Event() for _ in range(2)]      # upload into d_stage[b] finished
            self.consumed = [torch.cuda.Event() for _ in range(2)]    # set_spins has read d_stage[b]
            self.done = [torch.cuda.Event() for _ in range(2)]        # series of the step using h_obs[b] is on the host
        self.h2d_bytes_per_step = N
        self.d2h_bytes_per_step = 16 * S

    def run(self, inputs, consume=None, stream=None):
        """inputs: sequence of (h_in, sweep_counter), h_in a pinned int8 host tensor of N canonical spin values that must
        stay untouched until run returns.  consume(k, series) is called on the host, in step order, with the pinned
        int64 [S, 2] buffer holding step k's series (valid only during the call: copy what you keep).  Returns after the
        last series has been consumed; the lattice is left in the final state of the last step."""
        import torch

        lat = self.lat
        comp = torch.cuda.current_stream(lat.device) if stream is None else stream
        n = len(inputs)
        if n == 0:
            return
        self.copy_stream.wait_stream(comp)            # earlier work on the compute stream may still read d_stage
        lat.stage_spins_host(inputs[0][0], self.d_stage[0], self.copy_stream)
        self.staged[0].record(self.copy_stream)
        for k in range(n):
            b = k & 1
            comp.wait_event(self.staged[b])
            lat.set_spins(self.d_stage[b], inputs[k][1], stream=comp)      # layout conversion + full (B, M) reduction
            self.consumed[b].record(comp)
            if k + 1 < n:                                                    # next upload, behind this step's sweeps
                if k >= 1:
                    self.copy_stream.wait_event(self.consumed[b ^ 1])
                lat.stage_spins_host(inputs[k + 1][0], self.d_stage[b ^ 1], self.copy_stream)
                self.staged[b ^ 1].record(self.copy_stream)
            if k >= 2:                                                       # h_obs[b] still holds step k-2's series
                self.done[b].synchronize()
                if consume is not None:
                    consume(k - 2, self.h_obs[b])
            lat.sweep_record_host_async(self.S, self.h_obs[b], self.d_obs[b], stream=comp)
            self.done[b].record(comp)
        for k in range(max(n - 2, 0), n):
            self.done[k & 1].synchronize()
            if consume is not None:
                consume(k, self.h_obs[k & 1])
