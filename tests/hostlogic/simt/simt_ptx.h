// tests/hostlogic/simt/simt_ptx.h -- TEST INFRASTRUCTURE: host stand-ins for the inline-PTX helpers
// of csrc/search_staged.cu (same names, same signatures), included by that file in place of the
// PTX when KBMOD_SIMT_EMUL is defined.  mbarrier and TMA semantics as the PTX ISA states them:
//   * mbarrier: `pending` arrivals and a transaction count; the phase completes (parity flips,
//     pending reloads) when both reach zero; try_wait.parity(P) is true once the phase of parity
//     P has completed, i.e. when the current phase parity differs from P;
//   * cp.async.bulk.tensor (tiled, no swizzle): the box is written densely, elements outside the
//     tensor are zero-filled, the full box byte count is signalled on the mbarrier.  Checked here
//     because the hardware faults or rejects them: destination 128-byte aligned, innermost start
//     coordinate x element size a multiple of 16 bytes (measured on B200: "illegal instruction"
//     otherwise), box row a multiple of 16 bytes, box dims <= 256, strides multiples of 16 bytes.
#pragma once
// (no namespace and no includes here: search_staged.cu includes this file inside namespace kbmod,
// after <cuda.h> and <cuda_runtime.h> of this directory)

// shared-window address of a pointer into the CTA's shared-memory array (kbmod::smem_raw, owned by
// the test driver that links this translation unit)
extern unsigned char smem_raw[];
inline unsigned smem_u32(const void* p) {
    return simt::SMEM_BASE + (unsigned)(static_cast<const unsigned char*>(p) - smem_raw);
}

inline void mbar_touch(simt::MBar& b) {
    if (b.pending == 0 && b.tx == 0) { b.phase ^= 1u; b.pending = b.expected; }
    ++simt::S().steps;
}
inline simt::MBar& mbar_at(unsigned bar, bool must_exist = true) {
    if (bar & 7) simt::fatal("mbarrier address not 8-byte aligned");
    simt::smem_ptr(bar, 8, 8);
    simt::MBar& b = simt::S().bars[bar];
    if (must_exist && !b.init) simt::fatal("mbarrier used before mbarrier.init");
    return b;
}
inline void mbar_init(unsigned bar, unsigned count) {
    simt::MBar& b = mbar_at(bar, false);
    b = simt::MBar();
    b.expected = b.pending = (int)count;
    b.init = true;
}
inline void fence_mbar_init() {}
inline void mbar_arrive(unsigned bar) {
    simt::MBar& b = mbar_at(bar);
    if (b.pending <= 0) simt::fatal("mbarrier.arrive: more arrivals than the barrier expects in this phase");
    --b.pending;
    mbar_touch(b);
}
inline void mbar_arrive_expect_tx(unsigned bar, unsigned bytes) {
    simt::MBar& b = mbar_at(bar);
    if (b.pending <= 0) simt::fatal("mbarrier.arrive.expect_tx: more arrivals than expected");
    b.tx += bytes;
    --b.pending;
    mbar_touch(b);
}
inline void mbar_complete_tx(unsigned bar, unsigned bytes) {
    simt::MBar& b = mbar_at(bar);
    b.tx -= bytes;
    mbar_touch(b);
}
inline bool mbar_try_wait(unsigned bar, unsigned parity) {
    simt::MBar& b = mbar_at(bar);
    const bool ok = b.phase != (parity & 1u);
    simt::S().cur->where = "mbarrier.try_wait"; simt::S().cur->where_a = bar; simt::S().cur->where_b = parity;
    if (!ok) simt::yield();                    // let somebody else make progress before the next poll
    return ok;
}

inline void tma_load_3d(unsigned dst, const void* tmap, int c0, int c1, int c2, unsigned bar) {
    simt::State& s = simt::S();
    ++s.tma_loads;
    const simt::SimTensorMap m = *static_cast<const simt::SimTensorMap*>(tmap);
    if (m.magic != simt::TMAP_MAGIC) simt::fatal("TMA load through a tensor map that was never encoded");
    const unsigned bytes = m.box[0] * m.box[1] * m.box[2] * 4u;
    if ((dst & 127) || ((long long)c0 * 4) % 16 != 0) { ++s.tma_faults; }
    mbar_at(bar);
    auto copy = [=]() {
        const long long faults = simt::S().smem_faults;
        float* out = reinterpret_cast<float*>(simt::smem_ptr(dst, bytes, 128));
        if (simt::S().smem_faults != faults) { mbar_complete_tx(bar, bytes); return; }   // reported by the driver
        size_t k = 0;
        for (unsigned z = 0; z < m.box[2]; ++z)
            for (unsigned y = 0; y < m.box[1]; ++y)
                for (unsigned x = 0; x < m.box[0]; ++x, ++k) {
                    const long long gx = (long long)c0 + x, gy = (long long)c1 + y, gz = (long long)c2 + z;
                    float v = 0.0f;
                    if (gx >= 0 && gx < m.dims[0] && gy >= 0 && gy < m.dims[1] && gz >= 0 && gz < m.dims[2])
                        v = *reinterpret_cast<const float*>(static_cast<const char*>(m.base) + gz * m.strides[1] +
                                                            gy * m.strides[0] + gx * 4);
                    out[k] = v;
                }
        mbar_complete_tx(bar, bytes);
    };
    const int delay = simt::cfg().tma_delay > 0 ? (int)(simt::next_rand() % (unsigned)(simt::cfg().tma_delay + 1)) : 0;
    if (delay == 0) copy();
    else s.tma.push_back(simt::PendingTma{delay, copy});
}

template <int OFF>
inline unsigned long long lds64(unsigned a) {
    unsigned long long v;
    memcpy(&v, simt::smem_ptr(a + OFF, 8, 8), 8);
    return v;
}
inline void sts32(unsigned a, int v) { memcpy(simt::smem_ptr(a, 4, 4), &v, 4); }
inline int lds32(unsigned a) { int v; memcpy(&v, simt::smem_ptr(a, 4, 4), 4); return v; }
inline int4 lds128(unsigned a) { int4 v; memcpy(&v, simt::smem_ptr(a, 16, 16), 16); return v; }

