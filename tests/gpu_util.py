"""Helpers of the -m gpu parity tests: move seeded inputs to the device and run the C-ABI path."""
import numpy as np
import torch


def dev():
    return torch.device("cuda:0")


def to_dev(inp, key):
    """The tensor both sides consume: bf16 bit patterns when the case is bf16, else fp32 values."""
    a = getattr(inp, key)
    if a is None:
        return None
    if key in inp.bits:
        return torch.from_numpy(np.ascontiguousarray(inp.bits[key]).view(np.int16)).to(dev()).view(torch.bfloat16)
    return torch.from_numpy(np.ascontiguousarray(a)).to(dev())


def t32(a):
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev())


class TailRun:
    """Runs haste_forward_loss (+logits_out, dY unpack) and haste_backward for one Inputs object."""

    def __init__(self, inp, G, flags=0, label_offset=0, dw_dtype=None, loss_scale=0.0, B_max=None, want_logits=True):
        from paper_2606_01117_b200 import haste
        self.haste = haste
        self.inp = inp
        B, d = inp.X.shape
        L, K = inp.W.shape
        self.B, self.d, self.L, self.K, self.G = B, d, L, K, G
        dt = "bf16" if "X" in inp.bits else "f32"
        self.layer = haste.HasteLayer(d, L, G, K, B_max or max(B, 1), dt, dw_dtype=dw_dtype, label_offset=label_offset,
                                      loss_scale=loss_scale, flags=flags)
        self.X, self.W = to_dev(inp, "X"), to_dev(inp, "W")
        self.idx = t32(inp.idx)
        self.bias = t32(inp.bias)
        self.rowptr, self.col = t32(inp.rowptr), t32(inp.col)
        self.want_logits = want_logits

    def forward(self):
        B, L = self.B, self.L
        self.loss = torch.full((1,), float("nan"), device=dev())
        self.dY = self.layer.alloc_dy(B)
        self.dY.fill_(float("nan"))
        self.logits = torch.full((B, L), float("nan"), device=dev()) if self.want_logits else None
        self.layer.forward_loss(B, self.X, self.idx, self.W, self.bias, self.rowptr, self.col, loss=self.loss,
                                dY=self.dY, logits_out=self.logits)
        self.fwd_launches = self.layer.last_launch_count
        out = dict(loss=float(self.loss.item()))
        if self.want_logits:
            out["z"] = self.logits.cpu().numpy()
        dYf = torch.empty(B, L, device=dev())
        self.layer.dy_unpack(B, self.dY, dYf)
        out["dY"] = dYf.cpu().numpy()
        return out

    def backward(self, dY_BL=None, want_db=True, accumulate_into=None):
        """dY_BL: optional [B,L] fp32 numpy array fed through haste_dy_pack (stage-isolated parity)."""
        B, L, K, d = self.B, self.L, self.K, self.d
        if dY_BL is not None:
            self.dY = self.layer.alloc_dy(B)
            self.layer.dy_pack(B, t32(np.asarray(dY_BL, dtype=np.float32)), self.dY)
        dW = torch.full((L, K), float("nan"), dtype=self.layer.dw_tdtype, device=dev())
        db = torch.full((L,), float("nan"), device=dev()) if want_db else None
        if accumulate_into is not None:
            dX = t32(np.asarray(accumulate_into, dtype=np.float32)).clone()
        else:
            dX = torch.full((B, d), float("nan"), device=dev())
        self.layer.backward(B, self.X, self.idx, self.W, self.dY, dW=dW, dbias=db, dX=dX,
                            accumulate_dX=accumulate_into is not None)
        self.bwd_launches = self.layer.last_launch_count
        torch.cuda.synchronize()
        return dict(dW=dW.float().cpu().numpy(), db=None if db is None else db.cpu().numpy(), dX=dX.cpu().numpy())


def dy_rounded(inp, dY64):
    """dY as the library stores it: rounded once to the layer's dtype (bf16) or fp32."""
    from paper_2606_01117_b200 import synth
    a = np.asarray(dY64, dtype=np.float32)
    if "X" in inp.bits:
        return synth.round_bf16(a)[1].reshape(a.shape)
    return a
