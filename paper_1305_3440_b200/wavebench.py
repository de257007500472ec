import sys, os
sys.path.insert(0, os.environ.get("GF_PKG_ROOT", os.path.dirname(os.path.dirname(os.path.abspath(__file__)))))
import torch, gf_inputs as gi
import paper_1305_3440_b200 as gf
dev=torch.device("cuda:0")
dims=tuple(int(x) for x in os.environ.get("DIMS","32,32,32,32").split(","))
V=dims[0]*dims[1]*dims[2]*dims[3]
iters=int(os.environ.get("ITERS","400"))
variants=os.environ.get("VARIANTS","f64-18,f64-12,f32-18,f32-12").split(",")
lags=[int(x) for x in os.environ.get("LAGS","0").split(",")]
blocks=[int(x) for x in os.environ.get("BLOCKS","0").split(",")]
U=gi.torch_smooth_random_gauge(dims,0.6,1,device=dev)
def timeit(fld,prec,n):
    fld.iterate(20,gf.GF_OVERRELAX,1.7,0.0,prec); torch.cuda.synchronize()
    a,b=torch.cuda.Event(enable_timing=True),torch.cuda.Event(enable_timing=True)
    a.record(); fld.iterate(n,gf.GF_OVERRELAX,1.7,0.0,prec); b.record(); torch.cuda.synchronize()
    return a.elapsed_time(b)/n
for name in variants:
    pkey,recon=name.split("-"); recon=int(recon)
    prec=gf.GF_F64 if pkey=="f64" else gf.GF_F32
    cd=torch.complex128 if pkey=="f64" else torch.complex64
    nb=16*recon*(8 if pkey=="f64" else 4)
    fld=gf.GaugeField(dims,recon=recon,precisions=(pkey,),device=dev)
    fld.pack(U.to(cd).contiguous(),prec)
    def row(label,ms):
        su=V/(ms*1e-3)
        print("%s %-28s %.4f ms/iter %.3e su/s alg %.0f GB/s"%(name,label,ms,su,su*nb/1e9),flush=True)
    fld.set_wavefront(0); row("register kernel (default)",timeit(fld,prec,iters))
    fld.set_wavefront(3)
    # mode 3 also fuses in iterate; to time streamed half-sweeps use sweep() pairs
    def half(n):
        for _ in range(n):
            fld.sweep(0,gf.GF_OVERRELAX,1.7,0.0,prec); fld.sweep(1,gf.GF_OVERRELAX,1.7,0.0,prec)
    half(20); torch.cuda.synchronize()
    a,b=torch.cuda.Event(enable_timing=True),torch.cuda.Event(enable_timing=True)
    a.record(); half(iters); b.record(); torch.cuda.synchronize()
    row("streamed half-sweeps",a.elapsed_time(b)/iters)
    fld.set_wavefront(2)
    for bl in blocks:
        for lag in lags:
            fld.set_wave_tuning(lag,bl)
            row("fused lag=%d blocks=%d"%(lag,bl),timeit(fld,prec,iters))
    F,th=fld.measure(prec); print("   F=%.6f theta=%.3e"%(F[0],th[0]),flush=True)
    fld.close(); del fld; torch.cuda.empty_cache()
