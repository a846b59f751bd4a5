// schedule.cpp -- host-only helpers around the step: the paper's learning-rate recipe (row f3)
// and the parameter-range split used to shard the path across GPUs (row f4 / SURVEY.md 8(e)).
#include <cmath>

#include "internal.h"

// PAPER.md:70 (section 3): "(1) learning rate linear scaling by the ratio between effective
// batch size and baseline batch size. (2) linearly warmup the learning rate for the first 10
// epochs before annealing at a rate 1/sqrt(2) per epoch for the remaining epochs", with the
// worked example base batch 256 / lr 0.1, total batch 2560: "the learning rate increases by 0.1
// every epoch before reaching 1.0 at the 10th epoch".  Reading (R19): epochs are
// 1-based; epoch 1 runs at base_lr, epoch warmup_epochs at peak = base_lr * total/base, linear
// in between; epoch e > warmup_epochs runs at peak * (1/sqrt 2)^(e - warmup_epochs).
extern "C" int hadpsgd_lr_schedule(double base_lr, double base_batch, double total_batch,
                                   int warmup_epochs, int epoch, double* lr_out) {
    if (!lr_out || !(base_lr > 0.0) || !(base_batch > 0.0) || !(total_batch > 0.0) ||
        warmup_epochs < 1 || epoch < 1)
        return HADPSGD_INVALID_ARG;
    const double peak = base_lr * (total_batch / base_batch);
    if (epoch <= warmup_epochs) {
        *lr_out = warmup_epochs == 1
                      ? peak
                      : base_lr + (peak - base_lr) * static_cast<double>(epoch - 1) /
                                      static_cast<double>(warmup_epochs - 1);
    } else {
        *lr_out = peak * std::pow(0.5, 0.5 * static_cast<double>(epoch - warmup_epochs));
    }
    return HADPSGD_OK;
}

// Contiguous split of a P_padded-element buffer over `world` ranks in whole
// HADPSGD_SEG_ALIGN_ELEMS blocks: rank r owns [lo, hi).  The method is element-wise
// independent, so each rank runs the unchanged step on its range and no data-path collective
// is needed; only the diagnostics (sums over elements) are added across ranks.
extern "C" int hadpsgd_shard_range(int64_t P_padded, int world, int rank, int64_t* lo, int64_t* hi) {
    if (!lo || !hi || P_padded < 0 || world < 1 || rank < 0 || rank >= world ||
        P_padded % HADPSGD_SEG_ALIGN_ELEMS != 0)
        return HADPSGD_INVALID_ARG;
    const int64_t blocks = P_padded / HADPSGD_SEG_ALIGN_ELEMS;
    const int64_t base = blocks / world, extra = blocks % world;
    const int64_t b0 = rank * base + (rank < extra ? rank : extra);
    const int64_t b1 = b0 + base + (rank < extra ? 1 : 0);
    *lo = b0 * HADPSGD_SEG_ALIGN_ELEMS;
    *hi = b1 * HADPSGD_SEG_ALIGN_ELEMS;
    return HADPSGD_OK;
}
